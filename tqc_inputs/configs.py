"""The five BASELINE.json configs as seeded synthetic inputs.

cfg1-3 are circuits + gate->subcircuit assignments (the oracle turns them into
tensors by statevector simulation); cfg4-5 are synthetic cut networks with
i.i.d. random tensors, as the paper itself did for large runs ("random numbers
as the subcircuit output").
"""
from __future__ import annotations

import numpy as np

from . import circuits as C
from .network import Network
from .seeds import (STREAM_GATES, STREAM_LAYOUT, seed_for)

BATCH = {1: 2 ** 8, 2: 2 ** 20, 3: 2 ** 16, 4: 2 ** 18, 5: 1_000_000}
MODE = {1: "distribution", 2: "distribution", 3: "states", 4: "states", 5: "states"}


def cfg1_circuit() -> C.Circuit:
    """8 qubits, 2x4 grid, depth 6; columns {0,1} | {2,3}; the one crossing CZ
    (layer 2, qubits 1-2) goes to the left part => 2 wire cuts, 5 wires each."""
    circ = C.grid_random_circuit(2, 4, 6, seed_for(1, STREAM_GATES))
    C.assign_parts_by_column(circ, 4, [2], crossing_to="left")
    circ.name = "cfg1"
    return circ


def cfg2_circuit() -> C.Circuit:
    """20-qubit QAOA p=1 on a seeded random 3-regular graph, 3 parts of <= 10 wires."""
    circ = C.qaoa_regular_circuit(20, seed_for(2, STREAM_LAYOUT), seed_for(2, STREAM_GATES),
                                  m=3, w_max=10, k_target=6)
    circ.name = "cfg2"
    return circ


def cfg3_circuit() -> C.Circuit:
    """30-qubit hardware-efficient ansatz, 3 rotation layers / 2 CNOT ladders,
    parts {0-10 | 11-19 | 20-29} => K = 6, shapes (3,10) (6,9) (3,11)."""
    circ = C.hea_ladder_circuit(30, 3, seed_for(3, STREAM_GATES))
    C.assign_parts_by_qubit_ranges(circ, [11, 20])
    circ.name = "cfg3"
    return circ


def _adjacent_nodes(node_of_qubit, rows, cols):
    adj = set()
    for r in range(rows):
        for c in range(cols):
            a = node_of_qubit[r * cols + c]
            if c + 1 < cols:
                b = node_of_qubit[r * cols + c + 1]
                if a != b:
                    adj.add((min(a, b), max(a, b)))
            if r + 1 < rows:
                b = node_of_qubit[(r + 1) * cols + c]
                if a != b:
                    adj.add((min(a, b), max(a, b)))
    return sorted(adj)


def _network_from_blocks(n_qubits, node_of_qubit, adjacency, cut_pairs, rng, name, meta):
    m = max(node_of_qubit) + 1
    cuts, sub_cuts = [], [[] for _ in range(m)]
    for (a, b) in cut_pairs:
        up, down = (a, b) if rng.integers(0, 2) == 0 else (b, a)
        e = len(cuts)
        cuts.append((int(up), int(down)))
        sub_cuts[a].append(e)
        sub_cuts[b].append(e)
    # the caller's tensor axis order is a seeded shuffle of the incident cuts (exercises G6)
    for s in range(m):
        perm = rng.permutation(len(sub_cuts[s]))
        sub_cuts[s] = [sub_cuts[s][int(i)] for i in perm]
    sub_qubits = [[] for _ in range(m)]
    for q, s in enumerate(node_of_qubit):
        sub_qubits[s].append(q)
    net = Network(n_qubits, cuts, sub_cuts, sub_qubits, name=name, meta=dict(meta, adjacency=adjacency))
    net.validate()
    return net


def cfg4_network() -> Network:
    """64 qubits; 8 blocks of 2x4 qubits in a 4x2 arrangement; one cut on each of
    the 10 block adjacencies plus 4 more on seeded adjacencies (K = 14); o_s = 8."""
    rng = np.random.default_rng(seed_for(4, STREAM_LAYOUT))
    rows = cols = 8
    node_of_qubit = [(r // 2) * 2 + (c // 4) for r in range(rows) for c in range(cols)]
    adjacency = _adjacent_nodes(node_of_qubit, rows, cols)
    assert len(adjacency) == 10
    extra = [adjacency[int(i)] for i in rng.choice(len(adjacency), size=4, replace=False)]
    net = _network_from_blocks(64, node_of_qubit, adjacency, adjacency + extra, rng, "cfg4", {})
    for s in range(net.m):
        assert net.o(s) + net.u(s) <= 15          # w_s = o_s + u_s <= 15
    return net


def cfg5_network(c_lo: int = 5, c_hi: int = 8, max_per_adjacency: int = 3) -> Network:
    """196 qubits on a 14x14 grid; 49 blocks of 2x2 with 3 seeded blocks split into
    1x2 halves (52 nodes, sum o_s = 196); cuts laid on block adjacencies until each
    c_s reaches its seeded target in [c_lo, c_hi] (SURVEY.md G-cfg5 fallback)."""
    rng = np.random.default_rng(seed_for(5, STREAM_LAYOUT))
    rows = cols = 14
    split = sorted(int(i) for i in rng.choice(49, size=3, replace=False))
    node_of_block, next_id = {}, 0
    for b in range(49):
        if b in split:
            node_of_block[b] = (next_id, next_id + 1)
            next_id += 2
        else:
            node_of_block[b] = (next_id, next_id)
            next_id += 1
    assert next_id == 52
    node_of_qubit = []
    for r in range(rows):
        for c in range(cols):
            top, bottom = node_of_block[(r // 2) * 7 + (c // 2)]
            node_of_qubit.append(top if r % 2 == 0 else bottom)
    adjacency = _adjacent_nodes(node_of_qubit, rows, cols)
    m = 52
    target = rng.integers(c_lo, c_hi + 1, size=m)
    count = np.zeros(m, dtype=np.int64)
    per_adj = {p: 1 for p in adjacency}
    pairs = list(adjacency)
    for (a, b) in adjacency:
        count[a] += 1
        count[b] += 1
    while True:
        open_adj = [p for p in adjacency if count[p[0]] < target[p[0]] and count[p[1]] < target[p[1]]
                    and per_adj[p] < max_per_adjacency]
        if not open_adj:
            break
        p = open_adj[int(rng.integers(0, len(open_adj)))]
        pairs.append(p)
        per_adj[p] += 1
        count[p[0]] += 1
        count[p[1]] += 1
    net = _network_from_blocks(196, node_of_qubit, adjacency, pairs, rng, "cfg5",
                               {"split_blocks": split, "targets": [int(t) for t in target]})
    for s in range(net.m):
        assert net.o(s) + net.u(s) <= 15
    return net


def random_network(m: int, K: int, seed: int, o_lo: int = 0, o_hi: int = 3, connected: bool = True,
                   shuffle_qubits: bool = True) -> Network:
    """Small random cut network for tests: a random spanning tree (if connected)
    plus random extra cuts (parallel cuts allowed); random output-qubit ownership."""
    rng = np.random.default_rng(seed)
    pairs = []
    if connected and m > 1:
        order = rng.permutation(m)
        for i in range(1, m):
            j = int(order[int(rng.integers(0, i))])
            pairs.append((min(j, int(order[i])), max(j, int(order[i]))))
    while len(pairs) < K and m > 1:
        a, b = (int(x) for x in rng.choice(m, size=2, replace=False))
        pairs.append((min(a, b), max(a, b)))
    pairs = pairs[:max(K, len(pairs))]
    o = rng.integers(o_lo, o_hi + 1, size=m)
    n = int(o.sum())
    qubits = rng.permutation(n) if shuffle_qubits else np.arange(n)
    node_of_qubit = [0] * n
    pos = 0
    sub_q = []
    for s in range(m):
        qs = [int(q) for q in qubits[pos:pos + int(o[s])]]
        pos += int(o[s])
        sub_q.append(qs)
        for q in qs:
            node_of_qubit[q] = s
    cuts, sub_cuts = [], [[] for _ in range(m)]
    for (a, b) in pairs:
        up, down = (a, b) if rng.integers(0, 2) == 0 else (b, a)
        e = len(cuts)
        cuts.append((up, down))
        sub_cuts[a].append(e)
        sub_cuts[b].append(e)
    for s in range(m):
        perm = rng.permutation(len(sub_cuts[s]))
        sub_cuts[s] = [sub_cuts[s][int(i)] for i in perm]
    net = Network(n, cuts, sub_cuts, sub_q, name=f"rand_m{m}_K{len(cuts)}_s{seed}")
    net.validate()
    return net
