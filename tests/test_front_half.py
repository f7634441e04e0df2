"""Host-side tests of the front half (tqc_plan_from_circuit / tqc_plan_from_gates): circuit text -> DAG -> Greedy Graph
Growing (Alg. 2 / Alg. 3 / Table 1) -> cuts -> cut network -> plan, and the Eq. 4-6 cost report.
CPU only (no compute call).

Pins (none is the partitioner checking itself): Table 1 values worked by hand, the only feasible partition of
GHZ-3 under w_max = 2, the caps and the wire budget sum_s w_s = n + K recounted here from the gate
list, the oracle's own extraction O3 given the library's gate assignment (identical network and subcircuits), and the
paper's correctness claim on the result: the direct sum over the library-made network equals the uncut statevector
(P:195), with tensors built by the oracle.
"""
import os

import numpy as np
import pytest

import paper_2502_03445_b200 as tqc
from oracle import cost_model, cutting, reconstruct as R, statevector as sv
from tqc_inputs import circuits as C, configs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")

BENCHMARKS = {   # the paper's six benchmark kinds at desk size: (circuit, w_max, s_max)
    "supremacy": lambda: (C.grid_random_circuit(3, 4, 8, seed=5), 7, 9),
    "regular": lambda: (C.qaoa_graph_circuit(10, "regular", 6), 6, 8),
    "erdos": lambda: (C.qaoa_graph_circuit(7, "erdos", 7), 5, 6),
    "aqft": lambda: (C.aqft_circuit(8, seed=8), 6, 12),
    "wstate": lambda: (C.wstate_circuit(9), 4, 8),
    "ghz": lambda: (C.ghz_circuit(10), 4, 3),
}


def test_table1_merging_cost_values():
    assert tqc.tqc_cut_merging_cost(3, 10, 2, 20, 5, 10) == pytest.approx(0.3 + 0.1 + 0.5, abs=1e-15)      # x / T rows
    assert tqc.tqc_cut_merging_cost(3, 10, 2, 20, 12, 10) == pytest.approx(0.3 + 0.1 + 4 ** 2 + 1, abs=1e-12)   # 4^{x-T} + 1
    assert tqc.tqc_cut_merging_cost(3, 10, 2, 20, 10, 10) == pytest.approx(0.3 + 0.1 + 1.0, abs=1e-15)     # x = T is still "<= T"
    assert tqc.tqc_cut_merging_cost(11, 10, 2, 20, 5, 10) < 0                                               # not allowed
    assert tqc.tqc_cut_merging_cost(3, 10, 21, 20, 5, 10) < 0


def test_parser_round_trip_and_errors():
    circ = C.random_small_circuit(5, 6, 3)
    circ.gates += [("cp", (0.25,), (0, 3)), ("t", (), (1,)), ("tdg", (), (2,)), ("y", (), (3,)), ("z", (), (4,))]
    text = tqc.circuit_text(circ.n, circ.gates)
    a = tqc.tqc_plan_from_circuit(text, 5, 99)
    b = tqc.tqc_plan_from_gates(circ.n, circ.gates, 5, 99)
    assert a.serialize() == b.serialize() and a.cut_assignment(len(circ.gates)) == b.cut_assignment(len(circ.gates))
    for s in range(a.m):                                            # angles survive the text form bit for bit (repr)
        assert a.cut_subcircuit(s) == b.cut_subcircuit(s)
    bad = {"": "qubits", "qubits 2\ncx 0 0\n": "line 2", "qubits 2\nfoo 0\n": "line 2", "qubits 2\nh 0\n\nrx 0\n": "line 4",
           "qubits 2\nh 5\n": "line 2", "h 0\n": "line 1", "qubits 2\nh(0.3) 0\n": "line 2", "qubits 2\ncx 0\n": "line 2"}
    for text, where in bad.items():
        with pytest.raises(tqc.TqcError) as ei:
            tqc.tqc_plan_from_circuit(text, 4, 4)
        assert ei.value.code == -8 and where in str(ei.value), (text, str(ei.value))       # TQC_E_PARSE
    ok = tqc.tqc_plan_from_circuit("# comment\nqubits 2\n  h 0   # trailing\n\ncx 0 1\n", 2, 1)
    assert ok.m == 1 and ok.K == 0


def test_ghz3_has_one_feasible_partition():
    g = C.ghz_circuit(3)
    p = tqc.tqc_plan_from_gates(3, g.gates, 2, 1)                   # w_max = 2, s_max = 1: every cx alone
    net = p.cut_network()
    assert (net.m, net.K, net.cuts) == (2, 1, [(0, 1)])
    assert p.cut_assignment(3) == [0, 0, 1]
    s0, s1 = p.cut_subcircuit(0), p.cut_subcircuit(1)
    assert (s0["w"], s0["U_wires"], s0["D_wires"], s0["O_wires"]) == (2, [1], [], [0])       # qubit 1 is measured upstream ...
    assert (s1["w"], s1["U_wires"], s1["D_wires"], s1["O_wires"]) == (2, [], [0], [0, 1])    # ... and initialised downstream
    assert net.sub_qubits == [[0], [1, 2]]


def _recount(circ, part_of_gate):
    """w_s, s_s and the cuts recounted from the gate list alone: one wire per maximal same-part run of two-qubit gates on a
    qubit; a cut between consecutive runs."""
    runs, n2q, cuts = {}, {}, 0
    for q in range(circ.n):
        seq = [part_of_gate[i] for i, (_n, _p, qs) in enumerate(circ.gates) if len(qs) == 2 and q in qs]
        if not seq:
            runs[0] = runs.get(0, 0) + 1
            continue
        prev = None
        for p in seq:
            if p != prev:
                runs[p] = runs.get(p, 0) + 1
                cuts += prev is not None
            prev = p
    for i, (_n, _p, qs) in enumerate(circ.gates):
        if len(qs) == 2:
            n2q[part_of_gate[i]] = n2q.get(part_of_gate[i], 0) + 1
    return runs, n2q, cuts


@pytest.mark.parametrize("kind", sorted(BENCHMARKS))
def test_partition_meets_caps_and_matches_the_oracle_extraction(kind):
    circ, w_max, s_max = BENCHMARKS[kind]()
    plan = tqc.tqc_plan_from_gates(circ.n, circ.gates, w_max, s_max)
    parts = plan.cut_assignment(len(circ.gates))
    net = plan.cut_network()
    runs, n2q, cuts = _recount(circ, parts)
    assert net.K == cuts and net.m == max(parts) + 1 >= 2, (kind, net.m, net.K)
    for s in range(net.m):
        sub = plan.cut_subcircuit(s)
        assert 0 < sub["w"] == runs[s] <= w_max and sub["n2q"] == n2q.get(s, 0) <= s_max
        assert sub["w"] == len(sub["U_wires"]) + len(sub["O_wires"])
    assert sum(plan.cut_subcircuit(s)["w"] for s in range(net.m)) == circ.n + net.K              # wire budget
    # the oracle's O3 on the library's gate assignment: the identical cut network and subcircuits
    circ.parts = [parts[i] if len(qs) == 2 else None for i, (_n, _p, qs) in enumerate(circ.gates)]
    onet, osubs = cutting.extract(circ)
    assert (onet.n_qubits, list(onet.cuts), onet.sub_cuts, onet.sub_qubits) == (net.n_qubits, net.cuts, net.sub_cuts, net.sub_qubits)
    for s, osub in enumerate(osubs):
        sub = plan.cut_subcircuit(s)
        assert sub["w"] == osub.w and sub["gates"] == [(nm, tuple(p), tuple(w)) for (nm, p, w) in osub.gates]
        assert sub["D_wires"] == [w for (w, _e) in osub.D] and sub["U_wires"] == [w for (w, _e) in osub.U]
        assert sub["O_wires"] == [w for (w, _q) in osub.O]
        have = [e for (_w, e) in osub.D] + [e for (_w, e) in osub.U]
        assert sub["bond_pos"] == [onet.sub_cuts[s].index(e) for e in have]
    # determinism
    again = tqc.tqc_plan_from_gates(circ.n, circ.gates, w_max, s_max)
    assert again.cut_assignment(len(circ.gates)) == parts and again.serialize() == plan.serialize()
    # the paper's correctness claim on the library-made network: oracle tensors, direct sum == uncut statevector
    if net.K <= 8 and circ.n <= 12:
        _net, T64, _ = cutting.tensors_from_circuit(circ)
        bits = R.full_distribution_bits(circ.n)
        want = sv.uncut_probabilities(circ.n, circ.gates)
        got = R.direct_sum(onet, T64, bits) if net.K <= 6 else R.bucket_elimination(onet, T64, bits)
        assert np.abs(got - want).max() <= 1e-9


def test_loose_caps_keep_the_circuit_whole_and_tight_caps_are_infeasible():
    circ = C.grid_random_circuit(2, 3, 6, seed=2)
    n2q = sum(1 for g in circ.gates if len(g[2]) == 2)
    p = tqc.tqc_plan_from_gates(circ.n, circ.gates, circ.n, n2q, Q_max=1e9)
    assert p.m == 1 and p.K == 0 and p.cut_subcircuit(0)["w"] == circ.n
    with pytest.raises(tqc.TqcError) as ei:
        tqc.tqc_plan_from_gates(circ.n, circ.gates, 1, 5)           # one two-qubit gate already needs two wires
    assert ei.value.code == -4                                       # TQC_E_INFEASIBLE
    with pytest.raises(tqc.TqcError):
        tqc.tqc_plan_from_gates(circ.n, circ.gates, 0, 5)


def test_real_cfg4_and_cfg5_circuits_partition_under_the_paper_caps():
    """SURVEY G-cfg4 / G-cfg5: the partitioner on the REAL grid circuits (not used for timing): (m, K, max w) reported."""
    for rows, cols, depth in ((8, 8, 10), (14, 14, 8)):
        circ = C.grid_random_circuit(rows, cols, depth, seed=1)
        plan = tqc.tqc_plan_from_gates(circ.n, circ.gates, 15, 60)                    # <= 15 qubits, <= 60 gates
        net = plan.cut_network()
        subs = [plan.cut_subcircuit(s) for s in range(net.m)]
        assert max(x["w"] for x in subs) <= 15 and max(x["n2q"] for x in subs) <= 60
        assert sum(x["w"] for x in subs) == circ.n + net.K
        print(f"{rows}x{cols} depth {depth}: m = {net.m}, K = {net.K}, max w = {max(x['w'] for x in subs)}, "
              f"max cuts per subcircuit = {max(len(c) for c in net.sub_cuts)}, plan log2 cost = {plan.cost_log2:.1f}")


def _golden(name):
    out = {}
    for line in open(os.path.join(GOLDEN, name)):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            out[k] = float(v)
    return out


def test_cost_model_against_hand_worked_example_and_the_library():
    g = _golden("cost_model.txt")
    subs = [(1, 0, 3, 2), (0, 1, 3, 1)]
    assert cost_model.t_qpu(subs) == pytest.approx(g["t_qpu_clamped"], rel=1e-12)
    assert cost_model.t_qpu(subs, shots_log2=(1, 20)) == pytest.approx(g["t_qpu_unclamped"], rel=1e-12)
    assert cost_model.t_classical(2 * 144 * 1e6, 3.1e13) == pytest.approx(g["t_classical_fig5"], rel=1e-12)
    # the library's report on a cut circuit against the oracle-side formula fed with the library's own (u, d, w, t)
    circ, w_max, s_max = BENCHMARKS["supremacy"]()
    plan = tqc.tqc_plan_from_gates(circ.n, circ.gates, w_max, s_max)
    subs = [plan.cut_subcircuit(s) for s in range(plan.m)]
    udwt = [(len(x["U_wires"]), len(x["D_wires"]), x["w"], x["depth"]) for x in subs]
    rep = plan.cost_report(flops=3.1e13, n_states=1e6)
    assert rep["t_qpu"] == pytest.approx(cost_model.t_qpu(udwt), rel=1e-12)
    assert rep["c_tn_flop"] == pytest.approx(2.0 * 2.0 ** plan.cost_log2 * 1e6, rel=1e-9)
    assert rep["t_total"] == pytest.approx(cost_model.t_total(udwt, rep["c_tn_flop"], 3.1e13), rel=1e-12)
    assert rep["qpu_variants"] == sum(3 ** u * 4 ** d for (u, d, _w, _t) in udwt)
    # depths recounted here: ASAP layers of the subcircuit's local gate list
    for x in subs:
        lay = [0] * x["w"]
        for (_n, _p, ws) in x["gates"]:
            l = max(lay[w] for w in ws) + 1
            for w in ws:
                lay[w] = l
        assert x["depth"] == max(lay)
    # a plan that was not made from a circuit needs explicit depths
    net = configs.cfg4_network()
    p4 = tqc.tqc_plan(net)
    with pytest.raises(tqc.TqcError):
        p4.cost_report(flops=1e13)
    r4 = p4.cost_report(flops=1e13, n_states=2 ** 18, depth=[10] * net.m)
    d = [sum(1 for e in net.sub_cuts[s] if net.cuts[e][1] == s) for s in range(net.m)]
    u = [net.c(s) - d[s] for s in range(net.m)]
    assert r4["t_qpu"] == pytest.approx(cost_model.t_qpu([(u[s], d[s], u[s] + net.o(s), 10) for s in range(net.m)]), rel=1e-12)
