"""CPU oracle for the TensorQC reconstruction hot path — TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline /
`--impl reference` legs may import anything from here.  The product
(`paper_2502_03445_b200/`) never does, and shares no code, header, table or
helper with it; the only thing both sides consume is `tqc_inputs/` (seeded input
descriptions with none of the method's arithmetic).

Everything is float64 / complex128 and follows PAPER.md (arXiv 2502.03445) in
the paper's order and notation; `P:n` cites PAPER.md line n, `S:n` SPEC.md line n.

Modules
  statevector.py  O1 gates, O2 statevector simulation, O7 uncut probabilities
  cutting.py      O3 subcircuit extraction, O4 variants, O5 Pauli attribution -> T_s,
                  O5' an independent second construction of T_s
  reconstruct.py  O6 direct sum over all 4^K cut assignments (Eq. 1, with the
                  1/2 per cut of reading G1), Pi-1 rank-one closed form, O8 bucket elimination, O8' per-state pairwise
                  tensordot contraction along the oracle's own elimination order (the tier that checks cfg5)
  direct_sum.c    O6 again in plain C (depth-first odometer), the timed CPU baseline
  planner_ref.py  reference greedy contraction-order planner (rules P1-P6 of DESIGN.md)

Pins (tests/test_oracle_*.py, `-m "not gpu"`): closed forms (GHZ, W, |+> Pauli vector),
O6 == O7 on random cut circuits with complex gates, sum_x p = 1, partition and order
invariance, m=2 == A^T B (library GEMM), chain == matrix chain, einsum brute force,
slicing identity, rank-one closed form, the paper's 144 / 768 multiplication counts.
Parity status: every VALUE-producing function here is pinned.  planner_ref.plan and planner_ref.choose_slice_cuts
implement rules the paper does not fix (it delegates ordering to CoTenGra): they are pinned by the paper's
counts on the Fig. 5 network, by hand-worked step lists under rules P1-P6 (tests/golden/planner_steps.txt) and by
invariants, which cannot exclude every wrong tie-break - DESIGN.md section 3 says so ("plan parity: rules, not paper").
"""
