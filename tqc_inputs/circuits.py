"""Seeded circuit descriptions (gate NAMES, angles, operands) for configs 1-3.

No unitaries here: gate matrices are the oracle's business (oracle/statevector.py).
A circuit is a `Circuit(n, gates)` with gates = list of (name, params, qubits);
`parts[i]` gives the subcircuit id of two-qubit gate i (None for one-qubit
gates, which the oracle attaches to an adjacent two-qubit gate, PAPER.md
lines 590-593).

Gate names: h, rx, ry, rz (one angle), sx/sy/sw = exp(-i pi/4 P) for
P = X, Y, W=(X+Y)/sqrt2 (sqrt(X), sqrt(Y), sqrt(W) up to phase, reading G11),
cz, cx, rzz(gamma) = exp(-i gamma Z(x)Z); y, z, t, tdg; cp(lambda) = diag(1, 1, 1, e^{i lambda}).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class Circuit:
    n: int
    gates: list
    parts: list = field(default_factory=list)   # per gate: subcircuit id or None
    name: str = ""
    meta: dict = field(default_factory=dict)


_GRID_LAYER_PATTERN = [0, 4, 1, 5, 2, 6, 3, 7]


def grid_cz_layers(rows: int, cols: int, depth: int):
    """Reading G12: the 8-pattern CZ cycle; every grid edge fires once per 8 layers."""
    layers = []
    for layer in range(depth):
        pat = _GRID_LAYER_PATTERN[layer % 8]
        czs = []
        for r in range(rows):
            for c in range(cols):
                if c + 1 < cols and pat == (c + 2 * (r % 2)) % 4:
                    czs.append((r * cols + c, r * cols + c + 1))
                if r + 1 < rows and pat == 4 + ((r + 2 * (c % 2)) % 4):
                    czs.append((r * cols + c, (r + 1) * cols + c))
        layers.append(czs)
    return layers


def grid_random_circuit(rows: int, cols: int, depth: int, seed: int) -> Circuit:
    """Supremacy-style circuit: CZ layer then a random
    sqrt-gate from {sx, sy, sw} on every qubit, `depth` times (readings G11, G12)."""
    rng = np.random.default_rng(seed)
    n = rows * cols
    gates = []
    for czs in grid_cz_layers(rows, cols, depth):
        for (a, b) in czs:
            gates.append(("cz", (), (a, b)))
        picks = rng.integers(0, 3, size=n)
        for q in range(n):
            gates.append((("sx", "sy", "sw")[int(picks[q])], (), (q,)))
    return Circuit(n, gates, name=f"grid{rows}x{cols}d{depth}")


def assign_parts_by_column(circ: Circuit, cols: int, boundaries, crossing_to: str = "left") -> None:
    """Assign every two-qubit gate of a grid circuit to a column band.

    boundaries = ascending list of first columns of bands 1.. ; a gate whose two
    qubits fall in different bands goes to the left (lower) band.
    """
    def band(q):
        c = q % cols
        return sum(1 for b in boundaries if c >= b)
    parts = []
    for (name, _p, qs) in circ.gates:
        if len(qs) == 2:
            ba, bb = band(qs[0]), band(qs[1])
            parts.append(min(ba, bb) if crossing_to == "left" else max(ba, bb))
        else:
            parts.append(None)
    circ.parts = parts


def hea_ladder_circuit(n: int, layers: int, seed: int) -> Circuit:
    """Reading G14: `layers` rotation layers (RY then RZ on every qubit, angles
    U[0, 2pi)), with a CNOT(i, i+1), i = 0..n-2 ladder between consecutive layers."""
    rng = np.random.default_rng(seed)
    gates = []
    for layer in range(layers):
        ang = rng.random((n, 2)) * (2.0 * np.pi)
        for q in range(n):
            gates.append(("ry", (float(ang[q, 0]),), (q,)))
            gates.append(("rz", (float(ang[q, 1]),), (q,)))
        if layer + 1 < layers:
            for q in range(n - 1):
                gates.append(("cx", (), (q, q + 1)))
    return Circuit(n, gates, name=f"hea{n}l{layers}")


def assign_parts_by_qubit_ranges(circ: Circuit, firsts) -> None:
    """Gate on (a, b) goes to the band of its HIGHER qubit (so the boundary CNOT
    (10, 11) belongs to the middle part)."""
    def band(q):
        return sum(1 for f in firsts if q >= f)
    circ.parts = [band(max(qs)) if len(qs) == 2 else None for (_n, _p, qs) in circ.gates]


def random_regular_graph(n: int, degree: int, rng) -> list:
    """Seeded configuration-model pairing; rejects loops, multi-edges, disconnected graphs."""
    while True:
        stubs = np.repeat(np.arange(n), degree)
        rng.shuffle(stubs)
        edges = set()
        ok = True
        for i in range(0, len(stubs), 2):
            a, b = int(stubs[i]), int(stubs[i + 1])
            if a == b or (min(a, b), max(a, b)) in edges:
                ok = False
                break
            edges.add((min(a, b), max(a, b)))
        if not ok:
            continue
        adj = {v: set() for v in range(n)}
        for a, b in edges:
            adj[a].add(b)
            adj[b].add(a)
        seen, stack = {0}, [0]
        while stack:
            v = stack.pop()
            for w in adj[v]:
                if w not in seen:
                    seen.add(w)
                    stack.append(w)
        if len(seen) == n:
            return sorted(edges)


def _qaoa_cut_stats(edges, part_of, m):
    """cuts = number of distinct (wire, lower part) visits; wires per part."""
    visits = set()
    for a, b in edges:
        pa, pb = part_of[a], part_of[b]
        if pa != pb:
            lo = min(pa, pb)
            foreign = b if pa == lo else a
            visits.add((foreign, lo))
    wires = [0] * m
    for q, p in enumerate(part_of):
        wires[p] += 1
    for (_q, p) in visits:
        wires[p] += 1
    return len(visits), wires


def qaoa_partition_search(n: int, edges, m: int, w_max: int, rng, restarts: int = 30):
    """Seeded local search (single-vertex moves) for a vertex m-partition with few
    wire cuts under the wire cap; objective = 1000 * (excess wires) + cuts."""
    def score(part_of):
        k, wires = _qaoa_cut_stats(edges, part_of, m)
        if min(wires) == 0 or len(set(part_of)) < m:
            return (10 ** 9, k, wires)
        return (1000 * sum(max(0, w - w_max) for w in wires) + k, k, wires)
    best = None
    for _ in range(restarts):
        perm = rng.permutation(n)
        part_of = [0] * n
        for i, q in enumerate(perm):
            part_of[int(q)] = i * m // n
        cur = score(part_of)
        improved = True
        while improved:
            improved = False
            for q in range(n):
                for p in range(m):
                    old = part_of[q]
                    if p == old:
                        continue
                    part_of[q] = p
                    new = score(part_of)
                    if new[0] < cur[0]:
                        cur = new
                        improved = True
                    else:
                        part_of[q] = old
        if cur[0] < 1000 and (best is None or cur[1] < best[0]):
            best = (cur[1], list(part_of), cur[2])
    return best


def qaoa_regular_circuit(n: int, seed_graph: int, seed_angles: int, m: int = 3, w_max: int = 10,
                         k_target: int = 6, max_bumps: int = 64) -> Circuit:
    """Reading G13: H on all; rzz(gamma) per edge; rx(2 beta) per qubit; gamma, beta ~ U[0, pi].

    Edges are ordered by (assigned part, min, max) with a crossing edge assigned
    to the lower of its two parts, so each foreign wire visits a lower part
    before any of its home gates (ZZ gates commute; program order still defines
    the DAG).  The graph seed is bumped (+1000 each) until the partition search
    returns K <= k_target; the best seen is kept otherwise.
    """
    best = None
    for bump in range(max_bumps):
        rng = np.random.default_rng(seed_graph + 1000 * bump)
        edges = random_regular_graph(n, 3, rng)
        found = qaoa_partition_search(n, edges, m, w_max, rng)
        if found is None:
            continue
        if best is None or found[0] < best[0][0]:
            best = (found, edges, bump)
        if found[0] <= k_target:
            break
    (k, part_of, wires), edges, bump = best
    rng = np.random.default_rng(seed_angles)
    gamma, beta = (float(x) for x in rng.random(2) * np.pi)
    gates, parts = [], []
    for q in range(n):
        gates.append(("h", (), (q,)))
        parts.append(None)
    order = sorted(edges, key=lambda e: (min(part_of[e[0]], part_of[e[1]]), e[0], e[1]))
    for (a, b) in order:
        gates.append(("rzz", (gamma,), (a, b)))
        parts.append(min(part_of[a], part_of[b]))
    for q in range(n):
        gates.append(("rx", (2.0 * beta,), (q,)))
        parts.append(None)
    return Circuit(n, gates, parts, name=f"qaoa{n}",
                   meta={"edges": edges, "part_of": part_of, "K": k, "wires": wires,
                         "graph_seed_bump": bump, "gamma": gamma, "beta": beta})


def random_small_circuit(n: int, n_2q: int, seed: int, complex_gates: bool = True) -> Circuit:
    """Random test circuit with complex-amplitude one-qubit gates (needed to pin
    the Y-basis signs, reading G3) and random cz/cx/rzz between random pairs."""
    rng = np.random.default_rng(seed)
    gates = []
    for q in range(n):
        gates.append(("h", (), (q,)))
    ones = ("sx", "sy", "sw", "rz", "ry", "rx") if complex_gates else ("ry",)
    for _ in range(n_2q):
        a, b = (int(x) for x in rng.choice(n, size=2, replace=False))
        kind = ("cz", "cx", "rzz")[int(rng.integers(0, 3))]
        gates.append((kind, (float(rng.random() * np.pi),) if kind == "rzz" else (), (a, b)))
        for q in (a, b):
            nm = ones[int(rng.integers(0, len(ones)))]
            gates.append((nm, (float(rng.random() * 2 * np.pi),) if nm in ("rx", "ry", "rz") else (), (q,)))
    return Circuit(n, gates, name=f"rand{n}")


def assign_parts_random(circ: Circuit, m: int, seed: int) -> None:
    """Random gate->part assignment in which parts appear as contiguous runs of
    the two-qubit gate sequence merged with a random qubit-locality bias (test only)."""
    rng = np.random.default_rng(seed)
    home = rng.integers(0, m, size=circ.n)
    circ.parts = [int(home[qs[int(rng.integers(0, 2))]]) if len(qs) == 2 else None
                  for (_n, _p, qs) in circ.gates]


def hea_subcircuit(w: int = 12, d: int = 3, u: int = 3, seed: int = 250203445 + 4) -> dict:
    """Description of ONE synthetic subcircuit with the shape of cfg3's middle one (bench.py's `variants` row and its
    full-size parity test): three RY/RZ layers with a CX ladder after the first two, seeded angles; the first d wires
    begin at a downstream cut, the last u wires end at an upstream cut, the others at circuit outputs; bonds in
    (downstream..., upstream...) order.  Gate names and angles only: no arithmetic of the method."""
    rng = np.random.default_rng(seed)
    gates = []
    for layer in range(3):
        for q in range(w):
            gates.append(("ry", (float(rng.random() * 2 * np.pi),), (q,)))
            gates.append(("rz", (float(rng.random() * 2 * np.pi),), (q,)))
        if layer < 2:
            gates += [("cx", (), (q, q + 1)) for q in range(w - 1)]
    return dict(w=w, gates=gates, D_wires=list(range(d)), U_wires=list(range(w - u, w)), O_wires=list(range(w - u)),
                bond_pos=list(range(d + u)))


# ---- the paper's other benchmark families (section 7.2): gate lists only -----------------------
def ghz_circuit(n: int) -> Circuit:
    """GHZ-n: h 0; cx 0 1; cx 1 2; ... ("two dominating states").  Output law: 1/2 on 0..0 and on 1..1."""
    gates = [("h", (), (0,))] + [("cx", (), (q, q + 1)) for q in range(n - 1)]
    return Circuit(n, gates, name=f"ghz{n}")


def wstate_circuit(n: int) -> Circuit:
    """W-n ("n dominating states for a n-qubit benchmark"): x on qubit 0, then for k = 0..n-2 a rotation of qubit
    k+1 controlled on qubit k, RY(theta_k) with cos(theta_k / 2) = sqrt(1 / (n - k)), followed by cx(k+1, k).  The
    controlled RY is written with this package's gate names as ry(theta/2) t; cx c t; ry(-theta/2) t; cx c t.
    Output law: 1/n on each of the n one-hot bitstrings."""
    gates = [("x", (), (0,))]
    for k in range(n - 1):
        theta = 2.0 * float(np.arccos(np.sqrt(1.0 / (n - k))))
        c, t = k, k + 1
        gates += [("ry", (theta / 2.0,), (t,)), ("cx", (), (c, t)), ("ry", (-theta / 2.0,), (t,)), ("cx", (), (c, t)),
                  ("cx", (), (t, c))]
    return Circuit(n, gates, name=f"w{n}")


def aqft_circuit(n: int, degree: int | None = None, seed: int | None = None) -> Circuit:
    """Approximate QFT: for every target qubit j an h, then controlled phases cp(pi / 2^k) from qubit j + k,
    dropped when k > degree (default ceil(log2 n) + 2, the truncation the paper does not state).  No final swaps.
    With a seed the register first gets one ry(U[0, pi)) per qubit so that the output is not the flat distribution."""
    if degree is None:
        degree = int(np.ceil(np.log2(max(n, 2)))) + 2
    gates = []
    if seed is not None:
        rng = np.random.default_rng(seed)
        gates += [("ry", (float(rng.random() * np.pi),), (q,)) for q in range(n)]
    for j in range(n):
        gates.append(("h", (), (j,)))
        for k in range(1, n - j):
            if k <= degree:
                gates.append(("cp", (float(np.pi / 2 ** k),), (j + k, j)))
    return Circuit(n, gates, name=f"aqft{n}")


def qaoa_graph_circuit(n: int, kind: str, seed: int) -> Circuit:
    """The paper's Regular / Erdos benchmarks: one QAOA layer on a seeded random 3-regular graph ("regular") or
    G(n, 1/2) graph ("erdos"): h on all, rzz(gamma) per edge in ascending (min, max) order, rx(2 beta) on all; gamma, beta
    seeded in [0, pi) (reading G13)."""
    rng = np.random.default_rng(seed)
    if kind == "regular":
        edges = random_regular_graph(n, 3, rng)
    elif kind == "erdos":
        edges = [(a, b) for a in range(n) for b in range(a + 1, n) if rng.random() < 0.5]
    else:
        raise ValueError(kind)
    gamma, beta = (float(x) for x in rng.random(2) * np.pi)
    gates = [("h", (), (q,)) for q in range(n)]
    gates += [("rzz", (gamma,), (a, b)) for (a, b) in sorted(edges)]
    gates += [("rx", (2.0 * beta,), (q,)) for q in range(n)]
    return Circuit(n, gates, name=f"qaoa-{kind}{n}", meta={"edges": sorted(edges)})
