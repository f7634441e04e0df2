"""Pins for oracle/reconstruct.py, oracle/direct_sum.c and oracle/planner_ref.py — CPU only.

Pi-1 rank-one closed form, Pi-2 m=2 == library GEMM, Pi-3 chain == matrix chain,
Pi-4 brute-force einsum, Pi-5 slicing identity, Pi-6 distribution
sum, the paper's printed multiplication counts (144 / 768).
"""
import os

import numpy as np
import pytest

from oracle import planner_ref as P, reconstruct as R
from oracle.direct_sum_c import direct_sum_c
from tqc_inputs import configs, random_states, random_tensors, rank_one_tensors
from tqc_inputs.network import Network
from golden_planner import PLANNER_NETS, golden_planner_steps

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _golden(name):
    out = {}
    for line in open(os.path.join(GOLDEN, name)):
        if line.strip() and not line.startswith("#"):
            k, *v = line.split()
            out[k] = [int(x) for x in v]
    return out


def _fig5_network():
    # e1: 1-2, e2: 2-3, e3: 2-4, e4: 3-4 (0-based subcircuits 0..3, cuts 0..3)
    return Network(4, [(0, 1), (1, 2), (1, 3), (2, 3)], [[0], [0, 1, 2], [1, 3], [2, 3]], [[0], [1], [2], [3]])


def test_paper_multiplication_counts():
    g = _golden("fig5_counts.txt")
    net = _fig5_network()
    costs, kmax = R.multiplication_counts(net, [(0, 1), (4, 2), (5, 3)])       # ((1,2),3),4
    assert costs == g["steps_paper_order"] and sum(costs) == g["total_paper_order"][0]
    assert kmax == g["kmax_paper_order"][0]
    assert 4 ** net.K * (net.m - 1) == g["prior_method"][0]
    costs, _ = R.multiplication_counts(net, [(2, 3), (4, 1), (5, 0)])          # ((3,4),2),1
    assert costs == g["steps_alt_order"] and sum(costs) == g["total_alt_order"][0]
    assert g["prior_method"][0] / g["total_paper_order"][0] > 5                # "more than fivefold"


def test_m2_is_a_gemm():
    """Pi-2: two subcircuits => P = 2^{-K} A^T B, a library matmul."""
    net = Network(5, [(0, 1), (1, 0), (0, 1)], [[0, 1, 2], [0, 1, 2]], [[0, 1], [2, 3, 4]])
    T = random_tensors(net, 5)
    want = (T[0].astype(np.float64).T @ T[1].astype(np.float64)).reshape(-1) / 8.0
    bits = R.full_distribution_bits(5)
    assert np.allclose(R.direct_sum(net, T, bits), want, rtol=1e-13)
    assert np.allclose(direct_sum_c(net, T, bits)[0], want, rtol=1e-13)
    # axis order matters: permuting B's incident-cut order permutes its rows
    net2 = Network(5, net.cuts, [[0, 1, 2], [2, 0, 1]], net.sub_qubits)
    Bp = T[1].reshape(4, 4, 4, 8).transpose(2, 0, 1, 3).reshape(64, 8)         # axes (e2, e0, e1)
    assert np.allclose(R.direct_sum(net2, [T[0], Bp], bits), want, rtol=1e-13)
    assert np.allclose(direct_sum_c(net2, [T[0], Bp], bits)[0], want, rtol=1e-13)


def test_chain_is_a_matrix_chain():
    """Pi-3: A - B - C chain (config 3's shape) => 2^{-K} v_A^T W_B v_C."""
    net = Network(3, [(0, 1), (1, 0), (1, 2), (2, 1)], [[0, 1], [0, 1, 2, 3], [2, 3]], [[0], [1], [2]])
    T = [t.astype(np.float64) for t in random_tensors(net, 6)]
    bits = R.full_distribution_bits(3)
    want = np.zeros(8)
    for i, (a, b, c) in enumerate(bits):
        W = T[1][:, b].reshape(16, 16)
        want[i] = T[0][:, a] @ W @ T[2][:, c] / 16.0
    for got in (R.direct_sum(net, T, bits), direct_sum_c(net, T, bits)[0], R.bucket_elimination(net, T, bits)):
        assert np.allclose(got, want, rtol=1e-12)


def _einsum_brute_force(net, tensors, bits):
    """One einsum over explicit axes, per state."""
    out = np.zeros(bits.shape[0])
    keys = R.keys_from_bits(net, bits)
    for b in range(bits.shape[0]):
        args = []
        for s in range(net.m):
            v = np.asarray(tensors[s], dtype=np.float64)[:, keys[b, s]].reshape((4,) * net.c(s))
            args += [v, list(net.sub_cuts[s])]
        out[b] = np.einsum(*args, []) / 2.0 ** net.K
    return out


@pytest.mark.parametrize("seed", range(10))
def test_all_oracle_tiers_agree_on_tiny_networks(seed):
    """Pi-4 + order invariance."""
    m = 2 + seed % 4
    net = configs.random_network(m, (m - 1) + seed % 3, 50 + seed, o_lo=0, o_hi=2,
                                 connected=(seed % 5 != 4))
    if net.n_qubits == 0:
        net = configs.random_network(m, m, 50 + seed, o_lo=1, o_hi=2)
    T = random_tensors(net, 60 + seed)
    bits = random_states(net.n_qubits, 20, 70 + seed)
    want = _einsum_brute_force(net, T, bits)
    scale = np.abs(want).max()
    assert np.abs(R.direct_sum(net, T, bits) - want).max() <= 1e-12 * scale
    assert np.abs(direct_sum_c(net, T, bits)[0] - want).max() <= 1e-12 * scale
    assert np.abs(R.bucket_elimination(net, T, bits) - want).max() <= 1e-12 * scale
    assert np.abs(R.bucket_elimination(net, T, bits, order=list(range(net.K))[::-1]) - want).max() <= 1e-12 * scale
    for mode in (P.MODE_STATES, P.MODE_DISTRIBUTION):
        steps = P.step_pairs(P.plan(net, mode))
        assert np.abs(R.pairwise_contract(net, T, bits, steps) - want).max() <= 1e-12 * scale


@pytest.mark.parametrize("seed", range(4))
def test_rank_one_closed_form(seed):
    """Pi-1 against the literal sum (small K) and bucket elimination (K too large for 4^K)."""
    net = configs.random_network(4, 6, 80 + seed, o_lo=1, o_hi=3)
    T, g, a = rank_one_tensors(net, 90 + seed)
    bits = random_states(net.n_qubits, 16, 95 + seed)
    want = R.rank_one_closed_form(net, g, a, bits)
    assert np.allclose(R.direct_sum(net, T, bits), want, rtol=1e-13)
    assert np.allclose(direct_sum_c(net, T, bits)[0], want, rtol=1e-13)
    big = configs.random_network(12, 22, 180 + seed, o_lo=1, o_hi=2)
    T, g, a = rank_one_tensors(big, 190 + seed)
    bits = random_states(big.n_qubits, 8, 195 + seed)
    assert np.allclose(R.bucket_elimination(big, T, bits), R.rank_one_closed_form(big, g, a, bits), rtol=1e-12)


def test_slicing_identity():
    """Pi-5: fixing one cut to each of its 4 bases and summing reproduces the network (Fig. 6)."""
    net = configs.random_network(4, 5, 123, o_lo=1, o_hi=2)
    T = random_tensors(net, 124)
    bits = random_states(net.n_qubits, 12, 125)
    want = R.direct_sum(net, T, bits)
    e = 2
    total = np.zeros_like(want)
    keep = [x for x in range(net.K) if x != e]
    relabel = {x: i for i, x in enumerate(keep)}
    for basis in range(4):
        Ts, sub_cuts = [], []
        for s in range(net.m):
            t = np.asarray(T[s], dtype=np.float64)
            if e in net.sub_cuts[s]:
                ax = net.sub_cuts[s].index(e)
                t4 = t.reshape((4,) * net.c(s) + (-1,))
                t = np.take(t4, basis, axis=ax).reshape(4 ** (net.c(s) - 1), -1)
            Ts.append(t)
            sub_cuts.append([relabel[x] for x in net.sub_cuts[s] if x != e])
        sliced = Network(net.n_qubits, [net.cuts[x] for x in keep], sub_cuts, net.sub_qubits)
        total += R.direct_sum(sliced, Ts, bits) / 2.0          # the removed cut's 1/2
    assert np.allclose(total, want, rtol=1e-12)


def test_distribution_sum():
    """Pi-6: sum_x p(x) = 2^{-K} contract(sum_{x_s} T_s)."""
    net = configs.random_network(4, 5, 223, o_lo=1, o_hi=2)
    T = random_tensors(net, 224)
    p = R.direct_sum(net, T, R.full_distribution_bits(net.n_qubits))
    marg = Network(0, net.cuts, net.sub_cuts, [[] for _ in range(net.m)])
    Tm = [np.asarray(t, dtype=np.float64).sum(axis=1, keepdims=True) for t in T]
    tot = R.direct_sum(marg, Tm, np.zeros((1, 0), dtype=np.uint8))[0]
    assert np.isclose(p.sum(), tot, rtol=1e-12)


def test_c_direct_sum_on_cfg4_shape_prefix():
    """The C odometer at config-4 size (K = 14) on 2 states against bucket elimination."""
    net = configs.cfg4_network()
    assert (net.m, net.K, net.n_qubits) == (8, 14, 64)
    T = random_tensors(net, 1)
    bits = random_states(64, 2, 2)
    a, _ = direct_sum_c(net, T, bits)
    b = R.bucket_elimination(net, T, bits)
    assert np.allclose(a, b, rtol=1e-12)


def test_reference_planner_fixtures():
    net = _fig5_network()
    p = P.plan(net)
    costs, kmax = R.multiplication_counts(net, P.step_pairs(p))
    assert sum(costs) <= 144 and kmax <= 3 and p["kmax"] == kmax          # greedy is no worse than Fig. 5's order
    assert sum(costs) <= net.m * 4 ** kmax                                 # Eq. 2 bound
    assert [2 ** s["log2cost"] for s in p["steps"]] == costs
    # m = 2  =>  K_max = |E|
    net2 = Network(2, [(0, 1)] * 3, [[0, 1, 2], [0, 1, 2]], [[0], [1]])
    assert P.plan(net2)["kmax"] == 3
    # m > 3 connected => K_max < |E|
    for seed in range(5):
        big = configs.random_network(6, 9, 300 + seed, o_lo=1, o_hi=1)
        assert P.plan(big)["kmax"] < big.K
    # determinism and serialisation
    assert P.serialize(P.plan(net)) == P.serialize(P.plan(net))
    assert P.serialize(p)[:4] == b"TQCP"


@pytest.mark.parametrize("name", sorted(PLANNER_NETS))
def test_reference_planner_hand_worked_step_lists(name):
    """planner_ref.plan against step lists worked by hand under rules P1-P6 (tests/golden/planner_steps.txt): pins the
    memory score, its precedence over the cost exponent, both id tie-breaks, lhs = smaller id and merged parallel bonds."""
    net = PLANNER_NETS[name]()
    net.validate()
    assert P.plan(net)["steps"] == golden_planner_steps()[name]


@pytest.mark.parametrize("seed", range(6))
def test_tensordot_tier_and_order_search_against_direct_sum(seed):
    """O8' (contract_states_tensordot) and the seeded order search of O8 (order_trials > 0: the form the cfg5 GPU tests use)
    against the literal sum Pi-4 on tiny networks, parallel cuts and disconnected pieces included."""
    m = 3 + seed % 4
    net = configs.random_network(m, (m - 1) + seed % 4, 500 + seed, o_lo=0, o_hi=2, connected=(seed % 3 != 2))
    if net.n_qubits == 0:
        net = configs.random_network(m, m, 500 + seed, o_lo=1, o_hi=2)
    T = [t * (1 if seed % 2 else -1) ** np.arange(t.shape[1])[None, :] for t in random_tensors(net, 510 + seed)]   # signed
    bits = random_states(net.n_qubits, 12, 520 + seed)
    want = R.direct_sum(net, T, bits)
    scale = np.abs(want).max()
    assert np.abs(R.contract_states_tensordot(net, T, bits) - want).max() <= 1e-12 * scale
    assert np.abs(R.contract_states_tensordot(net, T, bits, order_trials=64) - want).max() <= 1e-12 * scale
    assert np.abs(R.bucket_elimination(net, T, bits, order_trials=64) - want).max() <= 1e-12 * scale
    order = R._elimination_order(net, trials=64)
    assert sorted(order) == list(range(net.K))                             # a permutation of the cut ids
    steps = R.pairwise_steps_from_elimination(net, order)
    assert np.abs(R.pairwise_contract(net, T, bits, steps + _join_rest(net, steps)) - want).max() <= 1e-12 * scale


def _join_rest(net, steps):
    """pairwise_contract multiplies leftover nodes itself; nothing to add (kept for clarity of the call above)."""
    return []


def test_tensordot_tier_at_cfg5_size_against_the_closed_form():
    """O8' at full cfg5 size (m = 52, K = 152) against Pi-1, the only exact pin there; distinct a_{s,e} per edge make any
    bond mix-up visible.  Also against O8 (bucket elimination) on a 22-cut network where both finish quickly."""
    net = configs.cfg5_network()
    T, g, a = rank_one_tensors(net, 55)
    bits = random_states(196, 3, 56)
    assert np.allclose(R.contract_states_tensordot(net, T, bits, order_trials=8), R.rank_one_closed_form(net, g, a, bits), rtol=1e-11)
    big = configs.random_network(12, 22, 181, o_lo=1, o_hi=2)
    Tb = random_tensors(big, 191)
    bb = random_states(big.n_qubits, 6, 196)
    assert np.allclose(R.contract_states_tensordot(big, Tb, bb), R.bucket_elimination(big, Tb, bb), rtol=1e-12)


def test_cfg5_network_shape_and_rank_one():
    net = configs.cfg5_network()
    assert net.m == 52 and net.n_qubits == 196
    assert sum(net.o(s) for s in range(52)) == 196
    assert all(2 <= net.o(s) <= 4 for s in range(52))
    p = P.plan(net)
    assert len(p["steps"]) == 51


@pytest.mark.parametrize("slice_cuts", [[2], [0, 3], [4, 1, 2]])
def test_sliced_sum_is_the_network(slice_cuts):
    """Pi-5 for oracle.reconstruct.sliced_sum: any set of sliced cuts (two on one tensor, parallel ones) sums back to Eq. 1."""
    net = configs.random_network(4, 6, 131, o_lo=1, o_hi=2)
    T = random_tensors(net, 132)
    bits = random_states(net.n_qubits, 10, 133)
    assert np.allclose(R.sliced_sum(net, T, bits, slice_cuts), R.direct_sum(net, T, bits), rtol=1e-12)
    small, Ts = R.slice_network(net, T, slice_cuts, [1] * len(slice_cuts))
    assert small.K == net.K - len(slice_cuts) and [t.shape[0] for t in Ts] == [4 ** small.c(s) for s in range(net.m)]


def _limits(net, mode, cuts):
    """Largest single-network input tensor and largest plan intermediate (log2 floats) with `cuts` sliced - recomputed here
    from the reduced network and the reference planner's steps."""
    small = P._without(net, cuts)
    big_in = max(2 * small.c(s) + small.o(s) for s in range(net.m))
    plan = P.plan(small, mode)
    bits = {s: small.o(s) for s in range(net.m)}
    worst = 0
    for t, st in enumerate(plan["steps"]):
        bits[net.m + t] = bits[st["lhs"]] + bits[st["rhs"]]
        worst = max(worst, 2 * (len(st["outer_lhs"]) + len(st["outer_rhs"])) + (bits[net.m + t] if mode else 0))
    return big_in, worst


@pytest.mark.parametrize("seed", range(8))
def test_choose_slice_cuts_reference_invariants(seed):
    """planner_ref.choose_slice_cuts (two-level slicing, PAPER.md 460-472): the chosen set meets both limits, nothing is
    sliced when nothing exceeds them, picks are distinct, and every pick was needed when it was made (the limit it serves
    was still violated by the picks before it)."""
    net = configs.random_network(3 + seed % 4, 6 + seed % 5, seed=900 + seed, o_lo=0, o_hi=4)
    for mode in (0, 1):
        in0, inter0 = _limits(net, mode, [])
        assert P.choose_slice_cuts(net, mode, in0, inter0) == []
        for lim_in, lim_inter in ((in0 - 2, 62), (62, max(inter0 - 3, 2)), (in0 - 2, max(inter0 - 4, 2))):
            S = P.choose_slice_cuts(net, mode, lim_in, lim_inter)
            if S is None:
                continue
            assert len(set(S)) == len(S) and all(0 <= e < net.K for e in S)
            got_in, got_inter = _limits(net, mode, S)
            assert got_in <= lim_in and got_inter <= lim_inter
            for k in range(len(S)):
                before_in, before_inter = _limits(net, mode, S[:k])
                assert before_in > lim_in or before_inter > lim_inter
