"""Heavy State Selection (section 4, Algorithm 1), float64.

Oracle code (test infrastructure): only tests/, __graft_entry__.smoke() and bench.py's CPU legs
may import it.  It follows Algorithm 1 line by line, in the paper's notation:

    x_j = {}                                            for all j                        (line 480)
    for each C_j, i:  ||p_{j,i}|| = sqrt(sum_e (p^e_{j,i})^2)                            (line 482)
                      add argmax_i ||p_{j,i}|| to x_j, remove that maximum               (lines 483-484)
    sort the remaining ||p_{j,i}|| in descending order                                   (line 486)
    while prod_j |x_j| < s_max:  pop ||p_{j,i}||, add i to x_j                           (lines 487-490)
    return x_j                                                                           (line 491)

p^e_{j,i} is the subcircuit tensor entry T_j[e, i] (edge permutation e = row, binary state i =
column).  Readings where the algorithm is silent (G18):
  - lines 483-484 sit inside the "for each C_j, i" loop but only make sense once per C_j (the
    arg max ranges over i): every subcircuit is seeded with its single heaviest state;
  - the seeds count toward prod_j |x_j|; the while-loop may overshoot s_max on its last addition
    and also ends when nothing is left to pop;
  - equal norms: smaller j first, then smaller i (the paper gives no rule; any total order gives a
    valid selection, this one makes it reproducible).

Pins (tests/test_oracle_hss.py): for a network with one subcircuit and no cut the selection is the
s_max most probable states (numpy argsort); a hand-worked two-subcircuit example; the selected set
is upward closed in the norm order apart from the seeds; prod_j |x_j| >= min(s_max, 2^n) with the
product below s_max before the last addition.
"""
from __future__ import annotations

import itertools

import numpy as np


def state_norms(tensor) -> np.ndarray:
    """||p_{j,i}|| for every binary state i of one subcircuit: the L2 norm over all edge
    permutations e (Alg. 1).  tensor is [4^{c_j}][2^{o_j}] (rows = e, columns = i)."""
    T = np.asarray(tensor, dtype=np.float64)
    out = np.zeros(T.shape[1], dtype=np.float64)
    for i in range(T.shape[1]):
        acc = 0.0
        for e in range(T.shape[0]):
            acc += T[e, i] * T[e, i]
        out[i] = np.sqrt(acc)
    return out


def state_norms_fast(tensor) -> np.ndarray:
    """Same quantity through numpy (used where the loop above would take minutes)."""
    T = np.asarray(tensor, dtype=np.float64)
    return np.sqrt((T * T).sum(axis=0))


def select(norms, s_max: int):
    """Algorithm 1 lines 480-491 on the per-subcircuit norm arrays.  Returns x_j as sorted lists."""
    m = len(norms)
    x = [set() for _ in range(m)]                                     # line 480
    remaining = []
    for j in range(m):
        nj = [float(v) for v in norms[j]]
        best = 0
        for i in range(1, len(nj)):                                   # arg max, first maximum wins
            if nj[i] > nj[best]:
                best = i
        x[j].add(best)                                                # line 483
        for i in range(len(nj)):                                      # line 484: the maximum is removed
            if i != best:
                remaining.append((nj[i], j, i))
    remaining.sort(key=lambda t: (-t[0], t[1], t[2]))                 # line 486
    pos = 0

    def product():
        p = 1
        for j in range(m):
            p *= len(x[j])
        return p

    while product() < s_max and pos < len(remaining):                 # line 487
        _, j, i = remaining[pos]                                      # line 488
        pos += 1
        x[j].add(i)                                                   # line 489
    return [sorted(s) for s in x]                                     # line 491


def expand(net, x):
    """The prod_j |x_j| composite n-qubit states the selection stands for,
    as a (B, n) 0/1 array; product order, subcircuit 0 slowest.  Bit order per reading G4: the
    first listed output qubit of a subcircuit is the most significant bit of i."""
    rows = []
    for combo in itertools.product(*x):
        bits = np.zeros(net.n_qubits, dtype=np.uint8)
        for j, key in enumerate(combo):
            qs = net.sub_qubits[j]
            for pos, q in enumerate(qs):
                bits[q] = (key >> (len(qs) - 1 - pos)) & 1
        rows.append(bits)
    if not rows:
        return np.zeros((0, net.n_qubits), dtype=np.uint8)
    return np.stack(rows)
