"""Pins for oracle/hss.py (Heavy State Selection, Alg. 1) and the host half of the
library's HSS entry points (tqc_hss_select / tqc_hss_expand need no GPU) — CPU only.

H-1  one subcircuit, no cut: the tensor is the probability vector, ||p_i|| = |p_i|, and the selection is the s_max
     most probable states (numpy argsort);
H-2  hand-worked example with integer norms (Pythagorean columns), every s_max from 1 to past the total;
H-3  the norm is numpy's column norm;
H-4  invariants on random networks: seeds present, the non-seed selection is a prefix of the descending norm
     order, prod |x_j| >= min(s_max, 2^n), and the product was below s_max before the last addition;
H-5  expansion: selecting everything enumerates every n-bit string exactly once, and the keys recovered from the
     expanded states by reconstruct.keys_from_bits (independent code, reading G4) are the product of the x_j;
H-6  the library's select/expand are bit-identical to the oracle, ties included, n > 64 included.
"""
import itertools

import numpy as np
import pytest

import paper_2502_03445_b200 as tqc
from oracle import hss as H, reconstruct as R
from tqc_inputs import configs, pack_states, random_tensors
from tqc_inputs.network import Network


def test_single_subcircuit_is_top_s():                                              # H-1
    rng = np.random.default_rng(11)
    p = rng.random(64)
    p /= p.sum()
    norms = H.state_norms(p[None, :])
    assert np.array_equal(norms, np.abs(p))
    order = np.argsort(-p, kind="stable")
    for s_max in (1, 2, 7, 63, 64, 1000):
        x = H.select([norms], s_max)
        assert x[0] == sorted(int(i) for i in order[:min(s_max, 64)])


def _hand_tensors():
    t0 = np.array([[3, 0], [4, 0], [0, 0], [0, 1]], dtype=np.float64)               # column norms 5, 1
    t1 = np.array([[1, 2, 0, 1], [2, 3, 0, 1], [2, 6, 0, 1], [0, 0, 2, 1]], dtype=np.float64)   # 3, 7, 2, 2
    return t0, t1


def test_hand_example():                                                            # H-2
    t0, t1 = _hand_tensors()
    norms = [H.state_norms(t0), H.state_norms(t1)]
    assert norms[0].tolist() == [5.0, 1.0] and norms[1].tolist() == [3.0, 7.0, 2.0, 2.0]
    # seeds {0}, {1}; then (C_1, 0) with 3, (C_1, 2) and (C_1, 3) with 2 (tie: smaller i first), (C_0, 1) with 1
    assert H.select(norms, 1) == [[0], [1]]
    assert H.select(norms, 2) == [[0], [0, 1]]
    assert H.select(norms, 3) == [[0], [0, 1, 2]]
    assert H.select(norms, 4) == [[0], [0, 1, 2, 3]]
    assert H.select(norms, 5) == [[0, 1], [0, 1, 2, 3]]                             # overshoots to 8
    assert H.select(norms, 100) == [[0, 1], [0, 1, 2, 3]]                           # everything, loop ends


def test_norm_is_column_norm():                                                     # H-3
    net = configs.random_network(4, 6, seed=5, o_lo=1, o_hi=4)
    for t in random_tensors(net, 9):
        want = np.linalg.norm(np.asarray(t, dtype=np.float64), axis=0)
        assert np.allclose(H.state_norms(t), want, rtol=1e-14, atol=0)
        assert np.allclose(H.state_norms_fast(t), want, rtol=1e-14, atol=0)


@pytest.mark.parametrize("seed", range(6))
def test_selection_invariants(seed):                                                # H-4
    net = configs.random_network(2 + seed % 4, 3 + seed, seed=100 + seed, o_lo=1, o_hi=4)
    norms = [H.state_norms_fast(t) for t in random_tensors(net, seed)]
    total = 2 ** net.n_qubits
    for s_max in (1, 2, 5, total // 3 + 1, total, 4 * total):
        x = H.select(norms, s_max)
        prod = int(np.prod([len(v) for v in x]))
        assert prod >= min(s_max, total)
        extra, left = [], []
        for j in range(net.m):
            seed_j = int(np.argmax(norms[j]))
            assert seed_j in x[j]
            for i in range(len(norms[j])):
                if i == seed_j:
                    continue
                (extra if i in x[j] else left).append((norms[j][i], j, i))
        if extra and left:
            assert min(e[0] for e in extra) >= max(l[0] for l in left)
        if extra:                                                                   # minimality of the stop
            last = min(extra, key=lambda t: (t[0], -t[1], -t[2]))
            sizes = [len(v) for v in x]
            sizes[last[1]] -= 1
            assert int(np.prod(sizes)) < s_max


def test_expand_enumerates_the_product():                                           # H-5
    net = configs.random_network(3, 4, seed=21, o_lo=1, o_hi=3)
    full = [list(range(2 ** net.o(j))) for j in range(net.m)]
    bits = H.expand(net, full)
    idx = (bits.astype(np.int64) << (net.n_qubits - 1 - np.arange(net.n_qubits))).sum(axis=1)
    assert sorted(idx.tolist()) == list(range(2 ** net.n_qubits))
    x = [[1], [0, 2 ** net.o(1) - 1], list(range(2 ** net.o(2)))[::2]]
    keys = R.keys_from_bits(net, H.expand(net, x))
    assert [tuple(r) for r in keys.tolist()] == list(itertools.product(*x))


@pytest.mark.parametrize("name", ["rand", "ties", "cfg4"])
def test_library_select_and_expand_match_oracle(name):                              # H-6
    rng = np.random.default_rng(3)
    if name == "cfg4":
        net = configs.cfg4_network()                                                # n > 64: two words per state
    else:
        net = configs.random_network(5, 7, seed=33, o_lo=0, o_hi=5)
    scores = [rng.random(2 ** net.o(j)).astype(np.float32) for j in range(net.m)]
    if name == "ties":
        scores = [np.round(s * 4).astype(np.float32) / 4 for s in scores]
    plan = tqc.tqc_plan(net, tqc.MODE_STATES)
    total = 2 ** net.n_qubits
    for s_max in (1, 3, 50, 4000, min(total, 1 << 16)):
        want = H.select([s.astype(np.float64) for s in scores], s_max)
        got = tqc.tqc_hss_select(plan, scores, s_max)
        assert [g.tolist() for g in got] == want
        if np.prod([float(len(v)) for v in want]) <= 1 << 17:
            states = tqc.tqc_hss_expand(plan, got)
            assert np.array_equal(states, pack_states(H.expand(net, want)))


def test_library_hss_argument_errors():
    net = configs.random_network(3, 3, seed=2, o_lo=1, o_hi=2)
    plan = tqc.tqc_plan(net, tqc.MODE_STATES)
    with pytest.raises(ValueError):
        tqc.tqc_hss_select(plan, [np.zeros(2, np.float32)], 4)
    with pytest.raises(tqc.TqcError):                                               # not loaded: TQC_E_STATE before any CUDA call
        tqc.binding._check(tqc.binding._lib.tqc_hss_scores(plan._h, 0, 1, None))
    with pytest.raises(tqc.TqcError):
        tqc.binding._check(tqc.binding._lib.tqc_hss_scores(plan._h, 7, 1, None))
