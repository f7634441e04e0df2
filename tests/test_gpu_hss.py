"""GPU parity for Heavy State Selection (Alg. 1) through the C ABI.

* tqc_hss_scores against oracle.hss.state_norms: fp32 sum of squares in 128 partial sums + a 7-level tree, so
  |d score| <= (cols/128 + 8) * 2^-24 * score;
* the selection made from GPU scores is a valid Alg. 1 selection up to that noise, and identical to the oracle's
  when the norms are separated by more than it;
* the whole pruned path: scores -> select -> expand -> tqc_contract_states equals the oracle's direct sum on the
  oracle's expanded states (|dp| <= 1e-5 max p, north_star).
"""
import numpy as np
import pytest
import torch

import paper_2502_03445_b200 as tqc
from oracle import hss as H
from oracle.direct_sum_c import direct_sum_c
from tqc_inputs import configs, random_tensors
from tqc_inputs.network import Network

pytestmark = pytest.mark.gpu


def _loaded(net, tensors):
    plan = tqc.tqc_plan(net, tqc.MODE_STATES)
    for s, t in enumerate(tensors):
        tqc.tqc_load_subcircuit_tensors(plan, s, np.ascontiguousarray(t, dtype=np.float32))
    return plan


def _gpu_scores(plan):
    out = [tqc.tqc_hss_scores(plan, s) for s in range(plan.m)]
    torch.cuda.synchronize()
    return [o.cpu().numpy() for o in out]


def _score_tol(net, s):
    return (4 ** net.c(s) / 128 + 8) * 2.0 ** -24


@pytest.mark.parametrize("case", ["rand_small", "rand_wide", "degenerate", "cfg4"])
def test_scores_match_oracle(case):
    if case == "rand_small":
        net = configs.random_network(5, 7, seed=41, o_lo=0, o_hi=5)
    elif case == "rand_wide":
        net = configs.random_network(3, 12, seed=42, o_lo=3, o_hi=9)              # up to 4^8 columns, several tiles of rows
    elif case == "degenerate":                                                      # o = 0 rows, c = 0 and c = 1 columns
        net = Network(3, [(0, 1)], [[0], [0], []], [[], [0, 1], [2]])
    else:
        net = configs.cfg4_network()
    tensors = [np.asarray(t, dtype=np.float32) for t in random_tensors(net, 7)]
    plan = _loaded(net, tensors)
    got = _gpu_scores(plan)
    for s in range(net.m):
        want = H.state_norms_fast(tensors[s])
        assert got[s].shape == want.shape
        assert np.all(np.abs(got[s] - want) <= _score_tol(net, s) * want + 1e-45), (case, s)


def test_selection_from_gpu_scores_is_valid_and_contracts():
    net = configs.random_network(4, 5, seed=43, o_lo=2, o_hi=5)
    tensors = [np.asarray(t, dtype=np.float32) for t in random_tensors(net, 8)]
    plan = _loaded(net, tensors)
    scores = _gpu_scores(plan)
    norms = [H.state_norms_fast(t) for t in tensors]
    tol = max(_score_tol(net, s) for s in range(net.m))
    for s_max in (1, 16, 300, 2000):
        x = tqc.tqc_hss_select(plan, scores, s_max)
        want = H.select(norms, s_max)
        assert int(np.prod([len(v) for v in x])) >= min(s_max, 2 ** net.n_qubits)
        extra, left = [], []
        for j in range(net.m):
            assert norms[j][x[j]].max() >= norms[j].max() * (1 - 2 * tol)         # the seed is a heaviest state
            sel = set(x[j].tolist())
            seed_j = int(np.argmax(scores[j]))
            for i in range(len(norms[j])):
                if i != seed_j:
                    (extra if i in sel else left).append(norms[j][i])
        if left and extra:
            assert min(extra) >= max(left) * (1 - 2 * tol)
        # random fp64 norms are separated by far more than the fp32 noise here: the selection is the oracle's
        gaps = np.diff(np.sort(np.concatenate(norms)))
        if gaps.min() > 4 * tol * np.concatenate(norms).max():
            assert [v.tolist() for v in x] == want
        states = tqc.tqc_hss_expand(plan, x)
        out = tqc.tqc_contract_states(plan, torch.from_numpy(states.view(np.int64)).cuda())
        torch.cuda.synchronize()
        bits = H.expand(net, [v.tolist() for v in x])
        ref = direct_sum_c(net, tensors, bits)[0]
        got = out.cpu().numpy().astype(np.float64)
        assert np.abs(got - ref).max() <= 1e-5 * np.abs(ref).max()


def test_scores_require_loaded_tensor():
    net = configs.random_network(3, 3, seed=2, o_lo=1, o_hi=2)
    plan = tqc.tqc_plan(net, tqc.MODE_STATES)
    with pytest.raises(tqc.TqcError):
        tqc.tqc_hss_scores(plan, 0)


@pytest.mark.parametrize("seed,s_max", [(0, 37), (1, 1000), (2, 1), (3, 20000)])
def test_product_structured_contraction(seed, s_max):
    """tqc_hss_contract (pruned output axes, one contraction) == the oracle's direct sum on the oracle's expansion ==
    tqc_contract_states on tqc_hss_expand's batch; |x_j| not powers of two, |x_j| = 1, o_j = 0 included."""
    net = configs.random_network(3 + seed, 6 + seed, seed=700 + seed, o_lo=0 if seed else 1, o_hi=5)
    tensors = [np.asarray(t, dtype=np.float32) for t in random_tensors(net, 710 + seed)]
    plan = _loaded(net, tensors)
    x = tqc.tqc_hss_select(plan, _gpu_scores(plan), s_max)
    assert plan.hss_cost_log2 < 0                                # nothing prepared yet
    got = tqc.tqc_hss_contract(plan, x)
    torch.cuda.synchronize()
    got = got.cpu().numpy().astype(np.float64)
    # the pruned plan's multiplication count: at least one multiplication per (padded) composite state and contraction step
    n_pad = np.prod([1 << int(np.ceil(np.log2(max(len(v), 1)))) for v in x], dtype=np.float64)
    assert plan.hss_cost_log2 >= np.log2(n_pad) - 1e-9
    bits = H.expand(net, [v.tolist() for v in x])
    assert got.shape == (bits.shape[0],)
    sample = np.arange(bits.shape[0]) if bits.shape[0] <= 4096 else np.random.default_rng(1).choice(bits.shape[0], 4096, replace=False)
    ref = direct_sum_c(net, tensors, bits[sample])[0]
    assert np.abs(got[sample] - ref).max() <= 1e-5 * np.abs(ref).max()
    states = tqc.tqc_hss_expand(plan, x)
    per_state = tqc.tqc_contract_states(plan, torch.from_numpy(states.view(np.int64)).cuda())
    torch.cuda.synchronize()
    assert np.abs(got - per_state.cpu().numpy()).max() <= 1e-5 * np.abs(ref).max()
    # a second selection with the same padded sizes reuses the pruned plan; a different one rebuilds it
    x2 = [np.sort(np.random.default_rng(2).permutation(1 << net.o(j))[:len(v)]).astype(np.int32) for j, v in enumerate(x)]
    got2 = tqc.tqc_hss_contract(plan, x2)
    torch.cuda.synchronize()
    ref2 = direct_sum_c(net, tensors, H.expand(net, [v.tolist() for v in x2])[:64])[0]
    assert np.abs(got2.cpu().numpy()[:64] - ref2).max() <= 1e-5 * max(np.abs(ref2).max(), np.abs(ref).max())
