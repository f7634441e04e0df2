"""GPU parity of the tensor-pipe step (step_tc_kernel: TMA-fed 3xTF32 tcgen05 MMAs, TMEM accumulators) against the
float64 direct sum of Eq. 1, on networks whose first contraction has large outer dimensions (M or N >= 128, K >= 32).
Same bar as everywhere: |dp| <= 1e-5 * max p; the 3xTF32 split is also compared with the fp32 FFMA path."""
import numpy as np
import pytest
import torch

import paper_2502_03445_b200 as tqc
from oracle.direct_sum_c import direct_sum_c
from tqc_inputs import pack_states, random_states, random_tensors
from tqc_inputs.network import Network

pytestmark = pytest.mark.gpu
TOL = 1e-5
KERNEL_TCGEN05 = 2


def _triangle(na, nb, ni, oa=5, ob=5, od=2, flip=False):
    """Subcircuits A, B, D: A-D share na cuts, B-D share nb, A-B share ni.  Contracting (A,B) first is a GEMM with
    M = 4^na, N = 4^nb, K = 4^ni per state; then a dot with D over 4^(na+nb)."""
    cuts, ca, cb, cd = [], [], [], []
    for _ in range(na):
        ca.append(len(cuts)); cd.append(len(cuts)); cuts.append((0, 2))
    for _ in range(nb):
        cb.append(len(cuts)); cd.append(len(cuts)); cuts.append((2, 1))
    for _ in range(ni):
        ca.append(len(cuts)); cb.append(len(cuts)); cuts.append((0, 1) if not flip else (1, 0))
    rng = np.random.default_rng(na * 100 + nb * 10 + ni)
    ca = [ca[i] for i in rng.permutation(len(ca))]            # caller axis order is arbitrary (G6)
    cb = [cb[i] for i in rng.permutation(len(cb))]
    cd = [cd[i] for i in rng.permutation(len(cd))]
    q = list(rng.permutation(oa + ob + od))
    net = Network(oa + ob + od, cuts, [ca, cb, cd], [[int(x) for x in q[:oa]], [int(x) for x in q[oa:oa + ob]],
                                                      [int(x) for x in q[oa + ob:]]], name=f"tri{na}{nb}{ni}")
    net.validate()
    return net


def _run(net, T, bits, **kw):
    plan = tqc.tqc_plan(net, tqc.MODE_STATES, **kw)
    for s, t in enumerate(T):
        tqc.tqc_load_subcircuit_tensors(plan, s, t)
    st = torch.from_numpy(pack_states(bits).view(np.int64)).cuda()
    out = tqc.tqc_contract_states(plan, st)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64), plan


@pytest.mark.parametrize("na,nb,ni,B", [(4, 2, 3, 67), (2, 4, 3, 33), (4, 3, 3, 40), (4, 4, 3, 9), (5, 2, 4, 21), (4, 2, 5, 16),
                                        (4, 5, 3, 5), (5, 4, 3, 3)])        # the last two: N >= 256, the wide-tile kernel
def test_tc_step_leaf_times_leaf(na, nb, ni, B):
    net = _triangle(na, nb, ni)
    T = random_tensors(net, 1000 + na * 100 + nb * 10 + ni)
    bits = random_states(net.n_qubits, B, 5)
    order = [(0, 1), (3, 2)]
    got, plan = _run(net, T, bits, order=order, batch_hint=4)
    assert plan.step(0)["kernel_class"] == KERNEL_TCGEN05
    want, _ = direct_sum_c(net, T, bits)
    err = np.abs(got - want).max() / want.max()
    assert err <= TOL, err
    ffma, plan2 = _run(net, T, bits, order=order, batch_hint=4, use_tcgen05=-1)
    assert plan2.step(0)["kernel_class"] != KERNEL_TCGEN05
    assert np.abs(got - ffma).max() / want.max() <= 3e-6


def _owned(pattern, ni, oa=1, ob=1, od=1):
    """A-B share ni cuts (the bond); the cuts to D are owned by A ('a') or B ('b') in ascending id order, which is the digit
    order of the result (last = lowest): the pattern decides which operand owns C's lowest offset bits."""
    cuts = [(0, 1)] * ni + [((0, 2) if ch == "a" else (1, 2)) for ch in pattern]
    ida = [ni + i for i, ch in enumerate(pattern) if ch == "a"]
    idb = [ni + i for i, ch in enumerate(pattern) if ch == "b"]
    net = Network(oa + ob + od, cuts, [list(range(ni)) + ida, list(range(ni)) + idb, ida + idb],
                  [list(range(oa)), list(range(oa, oa + ob)), list(range(oa + ob, oa + ob + od))], name="owned-" + pattern)
    net.validate()
    return net


@pytest.mark.parametrize("pattern,ni,B,signed", [("aaaabbbb", 3, 37, False),      # B owns the low digits: 8-byte stores
                                                 ("bbbbaaaa", 3, 21, True),       # A owns them: operands swapped by the launcher
                                                 ("abababab", 4, 18, True),       # interleaved digits
                                                 ("aaaaabbbb", 3, 5, False),      # M = 1024: several pair tiles per state
                                                 ("aaaabbbbb", 5, 3, False),      # N = 1024, K = 1024 (32 k-blocks per tile)
                                                 ("aaaabbbbb", 2, 29, True)])     # K = 16: one k-block, half of it zero fill
def test_pair_kernel_cta_group_2(pattern, ni, B, signed):
    """step_tc2_kernel (tcgen05 cta_group::2, 256 x 256 tiles over two SMs): both outer dimensions >= 256.  Ragged tile
    counts against the 74 clusters, both store orientations, signed values; against the float64 per-state contraction O8'
    and against the same plan on the FFMA kernels."""
    from oracle import reconstruct as R
    net = _owned(pattern, ni)
    rng = np.random.default_rng(len(pattern) * 10 + ni)
    T = [(rng.random(net.tensor_shape(s)) * (2 if signed else 1) - (1 if signed else 0)).astype(np.float32) for s in range(net.m)]
    bits = random_states(net.n_qubits, B, 11)
    got, plan = _run(net, T, bits, order=[(0, 1), (3, 2)], batch_hint=4)
    assert plan.step(0)["kernel_class"] == KERNEL_TCGEN05 and plan.pair_launch_count >= 1
    want = R.contract_states_tensordot(net, T, bits)
    scale = np.abs(want).max()
    assert np.abs(got - want).max() <= TOL * scale, np.abs(got - want).max() / scale
    ffma, plan2 = _run(net, T, bits, order=[(0, 1), (3, 2)], batch_hint=4, use_tcgen05=-1)
    assert plan2.pair_launch_count == 0
    assert np.abs(got - ffma).max() <= TOL * scale


def test_tc_step_with_batch_operand_and_signed_values():
    """4 subcircuits: (A,B) first (FFMA, small), then (AB, C) as a tensor-pipe step whose lhs is a per-state
    intermediate; signed values exercise the hi/lo split with cancellation."""
    # A-B: 2 cuts; A-C: 2 cuts, B-C: 1 cut (inner of step 2 = 3 cuts); A-D: 2, B-D: 2 (outer lhs = 4 cuts); C-D: 2 (outer rhs)
    cuts = [(0, 1), (1, 0), (0, 2), (2, 0), (1, 2), (0, 3), (3, 0), (1, 3), (3, 1), (2, 3), (3, 2)]
    sub = [[0, 1, 2, 3, 5, 6], [0, 1, 4, 7, 8], [2, 3, 4, 9, 10], [5, 6, 7, 8, 9, 10]]
    net = Network(14, cuts, sub, [[0, 1, 2, 3], [4, 5, 6, 7], [8, 9, 10, 11], [12, 13]], name="quad")
    net.validate()
    rng = np.random.default_rng(3)
    T = [(rng.random(net.tensor_shape(s)) * 2 - 1).astype(np.float32) for s in range(net.m)]
    bits = random_states(14, 50, 6)
    order = [(0, 1), (4, 2), (5, 3)]
    got, plan = _run(net, T, bits, order=order, batch_hint=4)
    assert plan.step(1)["kernel_class"] == KERNEL_TCGEN05
    want, _ = direct_sum_c(net, T, bits)
    assert np.abs(got - want).max() <= TOL * np.abs(want).max(), np.abs(got - want).max() / np.abs(want).max()


def test_warp_mma_paths_signed_values_and_ffma_agreement():
    """cfg4's plan has both warp-level 3xTF32 paths: a 16x16x16 step inside the fused chain kernel and table steps with a
    16-long bond and >= 2^10 rows per side (cross_mma_kernel).  Signed values (cancellation) against the direct sum, and
    against the same plan with use_tcgen05 = -1 / use_chain = -2 (fp32 FFMA tables, generic chain kernel)."""
    from tqc_inputs import configs
    net = configs.cfg4_network()
    rng = np.random.default_rng(17)
    T = [(rng.random(net.tensor_shape(s)) * 2 - 1).astype(np.float32) for s in range(net.m)]
    bits = random_states(net.n_qubits, 3000, 9)                         # ragged: not a multiple of 8 warps
    got, plan = _run(net, T, bits, batch_hint=1 << 18)
    from test_gpu_configs import require_specialised_chain
    require_specialised_chain(plan)
    ffma, _ = _run(net, T, bits, batch_hint=1 << 18, use_tcgen05=-1, use_chain=-2)
    want, _ = direct_sum_c(net, T, bits[:48])
    scale = np.abs(want).max()
    assert np.abs(got[:48] - want).max() <= TOL * scale, np.abs(got[:48] - want).max() / scale
    assert np.abs(ffma[:48] - want).max() <= TOL * scale
    assert np.abs(got - ffma).max() <= TOL * np.abs(ffma).max()


@pytest.mark.parametrize("oa,ob,na,nb,ni", [(3, 2, 2, 2, 2), (2, 3, 2, 2, 2), (4, 4, 1, 2, 3), (1, 5, 3, 1, 1)])
def test_cross_mma_tables_both_orientations_distribution_mode(oa, ob, na, nb, ni):
    """Distribution mode on a triangle A-B-D: step (A, B) is a cross-mode product with M' = 2^oa 4^na, N' = 2^ob 4^nb,
    K = 4^ni.  The cases put the >= 128 side on either operand (the launcher swaps them) and cover K = 4, 16, 64;
    (1, 5, 3, 1, 1) has K = 4 < 8 and must stay on the FFMA kernel.  Against the direct sum and the FFMA-only plan."""
    net = _triangle(na, nb, ni, oa=oa, ob=ob, od=1)
    T = [np.asarray(t, dtype=np.float32) for t in random_tensors(net, 40 + oa)]
    n = net.n_qubits
    idx = np.arange(2 ** n, dtype=np.int64)
    bits = ((idx[:, None] >> (n - 1 - np.arange(n))[None, :]) & 1).astype(np.uint8)
    want, _ = direct_sum_c(net, T, bits)
    outs = []
    for use_tc in (0, -1):
        plan = tqc.tqc_plan(net, tqc.MODE_DISTRIBUTION, order=[(0, 1), (3, 2)], use_tcgen05=use_tc)
        for s, t in enumerate(T):
            tqc.tqc_load_subcircuit_tensors(plan, s, t)
        out = tqc.tqc_contract_distribution(plan)
        torch.cuda.synchronize()
        outs.append(out.cpu().numpy().astype(np.float64))
        assert np.abs(outs[-1] - want).max() <= TOL * want.max()
        for pv in (1, 2):                                       # prefix slices: leaves addressed through a bit map
            part = tqc.tqc_contract_distribution(plan, pv, 2)
            torch.cuda.synchronize()
            w = want[pv << (n - 2):(pv + 1) << (n - 2)]
            assert np.abs(part.cpu().numpy() - w).max() <= TOL * want.max()
    assert np.abs(outs[0] - outs[1]).max() <= TOL * want.max()
