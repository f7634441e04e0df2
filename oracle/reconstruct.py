"""O6 direct sum (Eq. 1), the Pi-1 rank-one closed form, and O8 bucket elimination.

Oracle code (test infrastructure), float64.

The method reaches exactly the number the direct sum defines ("every sequence
ultimately yields the correct result"), so the oracle
is that definition written out:

    p(x) = 2^{-K} * sum_{k in {I,X,Y,Z}^K}  prod_{s=1..m}  T_s[ idx_s(k), x_s ]      (Eq. 1)

with the factor 1/2 per cut that the paper's Eq. 1 omits (reading G1: rho = 1/2 sum_P Tr(P rho) P).
idx_s(k) is the base-4 number whose digits are k_e for the cuts e incident on s, in the axis
order of the caller's tensor (net.sub_cuts[s], first = most significant; reading G6); x_s packs
the output bits of s (net.sub_qubits[s], first = MSB; reading G4).
"""
from __future__ import annotations

import itertools

import numpy as np


def keys_from_bits(net, bits: np.ndarray) -> np.ndarray:
    """x_s(b) for every state b and subcircuit s: (B, m) int64.  bits is (B, n) of 0/1."""
    B = bits.shape[0]
    keys = np.zeros((B, net.m), dtype=np.int64)
    for s in range(net.m):
        for q in net.sub_qubits[s]:
            keys[:, s] = (keys[:, s] << 1) | bits[:, q].astype(np.int64)
    return keys


def direct_sum(net, tensors, bits: np.ndarray) -> np.ndarray:
    """O6: the literal 4^K-term sum, vectorised over the batch of states only."""
    K, m = net.K, net.m
    keys = keys_from_bits(net, bits)
    T = [np.asarray(t, dtype=np.float64) for t in tensors]
    cols = [T[s][:, keys[:, s]] for s in range(m)]            # [4^{c_s}][B]: the x_s slices
    acc = np.zeros(bits.shape[0], dtype=np.float64)
    for k in itertools.product(range(4), repeat=K):           # all cut-basis assignments
        term = np.ones(bits.shape[0], dtype=np.float64)
        for s in range(m):
            idx = 0
            for e in net.sub_cuts[s]:
                idx = idx * 4 + k[e]
            term = term * cols[s][idx]
        acc += term
    return acc / (2.0 ** K)


def full_distribution_bits(n: int) -> np.ndarray:
    """All 2^n bitstrings in distribution order i = sum_q x_q 2^{n-1-q}."""
    idx = np.arange(2 ** n, dtype=np.int64)
    return ((idx[:, None] >> (n - 1 - np.arange(n))[None, :]) & 1).astype(np.uint8)


def rank_one_closed_form(net, g, a, bits: np.ndarray) -> np.ndarray:
    """Pi-1: if T_s[k, x] = g_s[x] prod_e a_{s,e}[k_e] then the sum of Eq. 1 factorises:
    p(x) = 2^{-K} prod_s g_s[x_s] prod_e (sum_k a_{up(e),e}[k] a_{down(e),e}[k])."""
    keys = keys_from_bits(net, bits)
    p = np.full(bits.shape[0], 2.0 ** (-net.K), dtype=np.float64)
    for s in range(net.m):
        p = p * np.asarray(g[s], dtype=np.float64)[keys[:, s]]
    for e, (up, down) in enumerate(net.cuts):
        p = p * float(np.dot(a[(up, e)], a[(down, e)]))
    return p


def _einsum(operands, out_labels):
    """np.einsum with arbitrary integer labels (remapped to 0..51 per call)."""
    remap = {}
    args = []
    for (v, lab) in operands:
        args += [v, [remap.setdefault(l, len(remap)) for l in lab]]
    return np.einsum(*args, [remap[l] for l in out_labels], optimize=len(operands) == 2)


def _elimination_order(net, trials: int = 0, seed: int = 0):
    """Order over cut ids for O8 (unrelated to the library's pairwise plan).  trials = 0: greedy
    min-size (eliminate the cut whose bucket product has the fewest labels, ties by cut id).
    trials > 0: the same greedy with seeded Gumbel noise on the score, repeated `trials` times;
    the order with the smallest total cost sum_e 4^{|labels of bucket e|} is kept.  Every
    elimination order yields the same value; only time and memory change."""
    def one_pass(rng, noise):
        groups = [set(es) for es in net.sub_cuts]
        remaining = set(range(net.K))
        order, cost = [], 0
        while remaining:
            best = None
            for e in sorted(remaining):
                touched = [g for g in groups if e in g]
                size = len(set().union(*touched)) - 1
                score = size + (noise * rng.gumbel() if noise > 0 else 0.0)
                if best is None or score < best[0]:
                    best = (score, e, size)
            e = best[1]
            cost += 4 ** (best[2] + 1)
            touched = [g for g in groups if e in g]
            merged = set().union(*touched) - {e}
            groups = [g for g in groups if e not in g] + [merged]
            remaining.discard(e)
            order.append(e)
        return cost, order
    best_cost, best_order = one_pass(None, 0.0)
    rng = np.random.default_rng(seed)
    for t in range(trials):
        cost, order = one_pass(rng, 0.3 + 0.1 * (t % 8))
        if cost < best_cost:
            best_cost, best_order = cost, order
    return best_order


def bucket_elimination(net, tensors, bits: np.ndarray, order=None, chunk: int = 64, order_trials: int = 0) -> np.ndarray:
    """O8: sum out one cut index at a time (variable elimination).  For cut e, multiply
    all current factors that carry e and sum over e; factors are float64 arrays with a
    leading batch axis.  Any elimination order gives the same value."""
    K, m = net.K, net.m
    if order is None:
        order = _elimination_order(net, trials=order_trials)
    keys = keys_from_bits(net, bits)
    T = [np.asarray(t, dtype=np.float64) for t in tensors]
    out = np.zeros(bits.shape[0], dtype=np.float64)
    BATCH = K                                                  # label of the batch axis
    for lo in range(0, bits.shape[0], chunk):
        kk = keys[lo:lo + chunk]
        nb = kk.shape[0]
        factors = []
        for s in range(m):
            v = T[s][:, kk[:, s]].T.reshape((nb,) + (4,) * net.c(s))
            factors.append((v, [BATCH] + list(net.sub_cuts[s])))
        for e in order:
            mine = [f for f in factors if e in f[1]]
            rest = [f for f in factors if e not in f[1]]
            labels = [BATCH] + sorted(set(l for f in mine for l in f[1]) - {e, BATCH})
            rest.append((_einsum(mine, labels), labels))
            factors = rest
        val = np.ones(nb, dtype=np.float64)
        for (v, lab) in factors:
            assert lab == [BATCH]
            val = val * v
        out[lo:lo + nb] = val / (2.0 ** K)
    return out


def pairwise_steps_from_elimination(net, order):
    """The pairwise order an elimination order over cut ids induces when parallel cuts are merged: take the
    cuts in `order`; a cut that is still open is held by exactly two current nodes, which are contracted over ALL the
    cuts they share.  Returns (lhs, rhs) node ids, leaves 0..m-1, step t creates m+t; a disconnected network leaves
    several nodes, multiplied at the end by the caller."""
    groups = {s: set(net.sub_cuts[s]) for s in range(net.m)}
    steps, nxt = [], net.m
    for e in order:
        holders = sorted(v for v, g in groups.items() if e in g)
        if len(holders) != 2:
            continue                                           # already summed together with a parallel cut
        a, b = holders
        steps.append((a, b))
        groups[nxt] = groups[a] ^ groups[b]
        del groups[a], groups[b]
        nxt += 1
    return steps


def contract_states_tensordot(net, tensors, bits: np.ndarray, order=None, order_trials: int = 0) -> np.ndarray:
    """O8' - the large-K tier that is fast enough for hundreds of cfg5 states: ONE STATE AT A TIME (no batch axis), the
    network is contracted pairwise along the order induced by the oracle's own elimination order (_elimination_order:
    greedy min-size with seeded noise, unrelated to the library's memory-score planner), each step a library
    `np.tensordot` over all cuts the two nodes share (multiply and sum over the shared indices; P:318-319
    parallel cuts are one bond).  Any order gives the same value.  float64 throughout."""
    if order is None:
        order = _elimination_order(net, trials=order_trials)
    steps = pairwise_steps_from_elimination(net, order)
    keys = keys_from_bits(net, bits)
    T = [np.asarray(t, dtype=np.float64) for t in tensors]
    out = np.zeros(bits.shape[0], dtype=np.float64)
    for b in range(bits.shape[0]):
        nodes = {s: (T[s][:, keys[b, s]].reshape((4,) * net.c(s)), list(net.sub_cuts[s])) for s in range(net.m)}
        for t, (u, v) in enumerate(steps):
            (va, la), (vb, lb) = nodes.pop(u), nodes.pop(v)
            shared = [l for l in la if l in lb]
            val = np.tensordot(va, vb, axes=([la.index(l) for l in shared], [lb.index(l) for l in shared]))
            nodes[net.m + t] = (val, [l for l in la if l not in shared] + [l for l in lb if l not in shared])
        p = 1.0
        for (val, lab) in nodes.values():
            assert lab == []
            p *= float(val)
        out[b] = p / (2.0 ** net.K)
    return out


def multiplication_counts(net, steps):
    """Per-step costs 4^{#inner + #outer} for a pairwise order given as
    (lhs, rhs) node ids (leaves 0..m-1, step t creates node m+t); returns (costs, K_max).
    Prior-method cost for comparison is 4^K (m-1)."""
    open_cuts = {s: set(net.sub_cuts[s]) for s in range(net.m)}
    costs, kmax = [], 0
    for t, (a, b) in enumerate(steps):
        union = open_cuts[a] | open_cuts[b]
        costs.append(4 ** len(union))
        kmax = max(kmax, len(union))
        open_cuts[net.m + t] = open_cuts[a] ^ open_cuts[b]
        del open_cuts[a], open_cuts[b]
    return costs, kmax


def pairwise_contract(net, tensors, bits: np.ndarray, steps) -> np.ndarray:
    """Contract along a given pairwise order in float64 (used for the order-invariance pin)."""
    keys = keys_from_bits(net, bits)
    B = bits.shape[0]
    BATCH = net.K
    nodes = {}
    for s in range(net.m):
        v = np.asarray(tensors[s], dtype=np.float64)[:, keys[:, s]].T.reshape((B,) + (4,) * net.c(s))
        nodes[s] = (v, [BATCH] + list(net.sub_cuts[s]))
    for t, (a, b) in enumerate(steps):
        (va, la), (vb, lb) = nodes.pop(a), nodes.pop(b)
        shared = (set(la) & set(lb)) - {BATCH}
        lo = [BATCH] + sorted((set(la) | set(lb)) - shared - {BATCH})
        nodes[net.m + t] = (_einsum([(va, la), (vb, lb)], lo), lo)
    val = np.ones(B, dtype=np.float64)
    for (v, lab) in nodes.values():
        assert lab == [BATCH]
        val = val * v
    return val / (2.0 ** net.K)


def slice_network(net, tensors, slice_cuts, assignment):
    """Index slicing (Fig. 6): fix every cut in slice_cuts to the basis given by `assignment`
    (same order).  Returns the smaller network (remaining cuts renumbered in order) and its tensors: each incident tensor
    keeps only the rows whose digit on the sliced axis equals the fixed basis."""
    from tqc_inputs.network import Network
    fixed = dict(zip(slice_cuts, assignment))
    keep = [e for e in range(net.K) if e not in fixed]
    relabel = {e: i for i, e in enumerate(keep)}
    Ts, sub_cuts = [], []
    for s in range(net.m):
        t = np.asarray(tensors[s], dtype=np.float64).reshape((4,) * net.c(s) + (-1,))
        index = tuple(fixed[e] if e in fixed else slice(None) for e in net.sub_cuts[s]) + (slice(None),)
        t = t[index]
        left = [e for e in net.sub_cuts[s] if e not in fixed]
        Ts.append(t.reshape(4 ** len(left), -1))
        sub_cuts.append([relabel[e] for e in left])
    return Network(net.n_qubits, [net.cuts[e] for e in keep], sub_cuts, net.sub_qubits), Ts


def sliced_sum(net, tensors, bits: np.ndarray, slice_cuts) -> np.ndarray:
    """The network as "a summation of smaller tensor networks": one direct sum per assignment of the sliced
    cuts' bases, each with its own 2^{-K'}; the 1/2 of every sliced cut (reading G1) is applied to the total."""
    acc = np.zeros(bits.shape[0], dtype=np.float64)
    for assignment in itertools.product(range(4), repeat=len(slice_cuts)):
        small, Ts = slice_network(net, tensors, list(slice_cuts), assignment)
        acc += direct_sum(small, Ts, bits)
    return acc / (2.0 ** len(slice_cuts))
