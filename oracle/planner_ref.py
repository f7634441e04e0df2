"""Reference greedy contraction-order planner — ORACLE-SIDE (test infrastructure).

The paper delegates ordering to CoTenGra; BASELINE.json's north_star
asks for a greedy planner whose plan is bit-identical between the library and this
reference.  Rules P1-P6 of DESIGN.md, all integer-valued:

P1 leaves are subcircuits 0..m-1; the node created at step t (0-based) has id m+t.
P2 candidates: all unordered pairs of live nodes sharing >= 1 cut; if none exist but
   more than one node is live (disconnected network) the single candidate is the pair
   of the two smallest live ids (outer product).
P3 two exact integers per candidate.  Cost exponent e(a,b) = 2*|E_a u E_b| in states mode
   (a step costs 4^{#inner+#outer} multiplications); + o_a + o_b in distribution
   mode (open output bits carried, reading G10).  Memory score
   sigma(a,b) = size(result) - size(a) - size(b), size(v) = 2^{w_v} 4^{|E_v|}, w_v = 0 in
   states mode and the carried output bits in distribution mode: the greedy objective of the
   order-search library the paper used (CoTenGra), which keeps the frontier of a 2-D
   network small where a pure min-cost rule grows one large tensor (reading P3).
P4 choose min sigma; tie -> smaller e; tie -> smaller min(id); tie -> smaller max(id).
P5 lhs = smaller id; all shared cuts are contracted together as one merged bond
   (P:318-319), digits in ascending cut id.
P6 K_max = max_t |E_a u E_b|; per-step log2 cost = e.

Serialisation (little-endian int32): 'TQCP', version 1, mode (0 states, 1 distribution),
n, m, K, then per step: lhs, rhs, #inner, #outer_lhs, #outer_rhs, log2cost, inner ids...,
outer_lhs ids..., outer_rhs ids... (each ascending); then K_max.
"""
from __future__ import annotations

import struct

MODE_STATES, MODE_DISTRIBUTION = 0, 1


def _sigma(open_cuts, obits, a, b, mode):
    wa = obits[a] if mode == MODE_DISTRIBUTION else 0
    wb = obits[b] if mode == MODE_DISTRIBUTION else 0
    r = len(open_cuts[a] ^ open_cuts[b])
    return (1 << (wa + wb + 2 * r)) - (1 << (wa + 2 * len(open_cuts[a]))) - (1 << (wb + 2 * len(open_cuts[b])))


def plan(net, mode: int = MODE_STATES):
    m = net.m
    open_cuts = {s: frozenset(net.sub_cuts[s]) for s in range(m)}
    obits = {s: net.o(s) for s in range(m)}
    steps = []
    t = 0
    while len(open_cuts) > 1:
        live = sorted(open_cuts)
        best = None
        for i, a in enumerate(live):
            for b in live[i + 1:]:
                if not (open_cuts[a] & open_cuts[b]):
                    continue
                e = 2 * len(open_cuts[a] | open_cuts[b])
                if mode == MODE_DISTRIBUTION:
                    e += obits[a] + obits[b]
                key = (_sigma(open_cuts, obits, a, b, mode), e, a, b)
                if best is None or key < best:
                    best = key
        if best is None:
            a, b = live[0], live[1]
            e = 2 * len(open_cuts[a] | open_cuts[b])
            if mode == MODE_DISTRIBUTION:
                e += obits[a] + obits[b]
            best = (0, e, a, b)
        _sig, e, a, b = best
        inner = sorted(open_cuts[a] & open_cuts[b])
        outer_a = sorted(open_cuts[a] - open_cuts[b])
        outer_b = sorted(open_cuts[b] - open_cuts[a])
        steps.append(dict(lhs=a, rhs=b, inner=inner, outer_lhs=outer_a, outer_rhs=outer_b, log2cost=e))
        new = m + t
        open_cuts[new] = open_cuts[a] ^ open_cuts[b]
        obits[new] = obits[a] + obits[b]
        del open_cuts[a], open_cuts[b]
        t += 1
    kmax = max([len(s["inner"]) + len(s["outer_lhs"]) + len(s["outer_rhs"]) for s in steps], default=0)
    return dict(mode=mode, n=net.n_qubits, m=m, K=net.K, steps=steps, kmax=kmax)


def serialize(p) -> bytes:
    words = [p["mode"], p["n"], p["m"], p["K"]]
    for s in p["steps"]:
        words += [s["lhs"], s["rhs"], len(s["inner"]), len(s["outer_lhs"]), len(s["outer_rhs"]), s["log2cost"]]
        words += s["inner"] + s["outer_lhs"] + s["outer_rhs"]
    words.append(p["kmax"])
    return b"TQCP" + struct.pack("<i", 1) + struct.pack(f"<{len(words)}i", *words)


def step_pairs(p):
    return [(s["lhs"], s["rhs"]) for s in p["steps"]]


def _without(net, slice_cuts):
    """The network with the given cuts removed (remaining cuts renumbered in order) - structure only."""
    from tqc_inputs.network import Network
    gone = set(slice_cuts)
    keep = [e for e in range(net.K) if e not in gone]
    relabel = {e: i for i, e in enumerate(keep)}
    return Network(net.n_qubits, [net.cuts[e] for e in keep],
                   [[relabel[e] for e in net.sub_cuts[s] if e not in gone] for s in range(net.m)], net.sub_qubits)


def choose_slice_cuts(net, mode, max_log2_input_floats, max_log2_intermediate_floats):
    """Two-level slicing, the reading written in include/tqc.h / DESIGN.md G19.
    Level 1: while a tensor of one sub-network exceeds the input limit, slice the most size-reducing cut among those
    touching an oversize tensor (its two tensors compared larger first, then smaller; tie: smaller id).
    Level 2: while the plan's largest intermediate exceeds its limit, slice the cut that leaves the smallest largest
    intermediate, then the smallest exact multiplication count, then the smaller id.  Returns None when infeasible."""
    S = []
    while True:
        small = _without(net, S)
        lg = [2 * small.c(s) + small.o(s) for s in range(net.m)]
        if max(lg) <= max_log2_input_floats:
            break
        best = None
        for e in range(net.K):
            if e in S:
                continue
            a, b = lg[net.cuts[e][0]], lg[net.cuts[e][1]]
            if max(a, b) <= max_log2_input_floats:
                continue
            key = (-max(a, b), -min(a, b), e)
            if best is None or key < best:
                best = key
        if best is None:
            return None
        S.append(best[2])

    def score(cuts):
        small = _without(net, cuts)
        p = plan(small, mode)
        bits = {s: small.o(s) for s in range(net.m)}
        worst = 0
        for t, st in enumerate(p["steps"]):
            bits[net.m + t] = bits[st["lhs"]] + bits[st["rhs"]]
            size = 2 * (len(st["outer_lhs"]) + len(st["outer_rhs"])) + (bits[net.m + t] if mode == MODE_DISTRIBUTION else 0)
            worst = max(worst, size)
        return worst, sum(1 << st["log2cost"] for st in p["steps"])

    while True:
        worst, _ = score(S)
        if worst <= max_log2_intermediate_floats:
            return S
        best = None
        for e in range(net.K):
            if e in S:
                continue
            w, c = score(S + [e])
            key = (w, c, e)
            if best is None or key < best:
                best = key
        if best is None:
            return None
        S.append(best[2])
