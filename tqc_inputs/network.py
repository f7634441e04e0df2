"""Cut-network description and raw random inputs (tensor values, bitstrings).

Notation (section 2.1; SURVEY.md section 8 "Notation"):
n qubits, m subcircuits, K = |E| wire cuts; subcircuit s touches the cut set
E_s (c_s = |E_s| cuts, d_s of them downstream ends) and carries o_s output
qubits of the original circuit.  Its tensor T_s has 4^{c_s} x 2^{o_s} entries.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class Network:
    """A cut network: which subcircuit touches which cut, and which output qubits it owns.

    cuts[e] = (up_sub, down_sub): cut e leaves subcircuit up_sub (measured end)
        and enters subcircuit down_sub (initialised end).  Cut id = index.
    sub_cuts[s]: incident cut ids of subcircuit s IN THE AXIS ORDER OF THE
        CALLER'S TENSOR: T_s is [4^{c_s}][2^{o_s}] row-major and the first listed
        cut is the most significant base-4 digit of the row index (reading G6).
    sub_qubits[s]: the global output qubits of s; the first listed is the MSB of
        the packed key x_s (reading G4: ascending global id is the convention
        the generators use, but any order is legal).
    """
    n_qubits: int
    cuts: list
    sub_cuts: list
    sub_qubits: list
    name: str = ""
    meta: dict = field(default_factory=dict)

    @property
    def m(self) -> int:
        return len(self.sub_cuts)

    @property
    def K(self) -> int:
        return len(self.cuts)

    def c(self, s: int) -> int:
        return len(self.sub_cuts[s])

    def o(self, s: int) -> int:
        return len(self.sub_qubits[s])

    def d(self, s: int) -> int:
        return sum(1 for e in self.sub_cuts[s] if self.cuts[e][1] == s)

    def u(self, s: int) -> int:
        return sum(1 for e in self.sub_cuts[s] if self.cuts[e][0] == s)

    def tensor_shape(self, s: int):
        return (4 ** self.c(s), 2 ** self.o(s))

    def validate(self) -> None:
        m, K = self.m, self.K
        assert len(self.sub_qubits) == m
        seen = [0] * K
        for s in range(m):
            assert len(set(self.sub_cuts[s])) == len(self.sub_cuts[s])
            for e in self.sub_cuts[s]:
                assert 0 <= e < K and s in self.cuts[e]
                seen[e] += 1
        assert all(v == 2 for v in seen), "every cut joins exactly two subcircuits"
        for (a, b) in self.cuts:
            assert a != b and 0 <= a < m and 0 <= b < m
        allq = [q for qs in self.sub_qubits for q in qs]
        assert sorted(allq) == list(range(self.n_qubits)), "sum_s o_s = n, each qubit once"


def random_tensors(net: Network, seed: int) -> list:
    """Reading G7: i.i.d. U[0,1) fp32, times the exact power of two 2^{1-d_s}."""
    rng = np.random.default_rng(seed)
    out = []
    for s in range(net.m):
        t = rng.random(net.tensor_shape(s), dtype=np.float32)
        t *= np.float32(2.0 ** (1 - net.d(s)))
        out.append(t)
    return out


_DYADIC = np.array([0.5, 0.75, 1.0, 1.5], dtype=np.float64)


def rank_one_tensors(net: Network, seed: int, signed: bool = False):
    """Factor vectors for the rank-one closed-form pin.

    Returns (tensors, g, a): g[s] is a length-2^{o_s} vector, a[(s, e)] a
    length-4 vector, all entries drawn from {0.5, 0.75, 1, 1.5} (two significant
    bits) so that T_s[k, x] = g_s[x] * prod_e a_{s,e}[k_e] is EXACT in fp32 for
    c_s <= 10.  The tensors are the plain outer products; the closed form that
    uses g and a lives with the oracle.  signed = True: every factor vector and
    every g entry gets a random overall sign (results of both signs, no
    cancellation), and on every eighth cut ONE entry of the downstream vector is
    flipped - the one with the smallest product - so that those bond sums cancel
    partially with a bounded condition number (sum |terms| / |sum| <= 2).  Fully
    random entry signs would make the value 10^60 times smaller than its terms at
    cfg5 size: any fp32 evaluation, FFMA or tensor pipe alike, then loses three
    more digits, which is a property of the data, not of a kernel.
    """
    rng = np.random.default_rng(seed)
    g, a = [], {}
    for s in range(net.m):
        g.append(_DYADIC[rng.integers(0, 4, size=2 ** net.o(s))])
        for e in net.sub_cuts[s]:
            a[(s, e)] = _DYADIC[rng.integers(0, 4, size=4)]
    if signed:
        for s in range(net.m):
            g[s] = g[s] * rng.choice([-1.0, 1.0], size=g[s].shape)
            for e in net.sub_cuts[s]:
                a[(s, e)] = a[(s, e)] * float(rng.choice([-1.0, 1.0]))
        for e, (up, down) in enumerate(net.cuts):
            if e % 8 == 0:
                k = int(np.argmin(np.abs(a[(up, e)] * a[(down, e)])))
                a[(down, e)][k] = -a[(down, e)][k]
    tensors = []
    for s in range(net.m):
        row = np.ones(1, dtype=np.float64)
        for e in net.sub_cuts[s]:          # first listed cut = most significant digit
            row = np.multiply.outer(row, a[(s, e)]).reshape(-1)
        t = np.multiply.outer(row, g[s])
        t32 = t.astype(np.float32)
        assert np.array_equal(t32.astype(np.float64), t)
        tensors.append(t32)
    return tensors, g, a


def random_states(n_qubits: int, count: int, seed: int) -> np.ndarray:
    """`count` bitstrings uniform over {0,1}^n, as a (count, n) uint8 array of bits."""
    rng = np.random.default_rng(seed)
    return rng.integers(0, 2, size=(count, n_qubits), dtype=np.uint8)


def pack_states(bits: np.ndarray) -> np.ndarray:
    """Reading G5: ceil(n/64) u64 words per state, qubit q at word q//64, bit q%64."""
    count, n = bits.shape
    words = (n + 63) // 64
    out = np.zeros((count, words), dtype=np.uint64)
    for q in range(n):
        out[:, q // 64] |= bits[:, q].astype(np.uint64) << np.uint64(q % 64)
    return out


def index_to_bits(idx: np.ndarray, n_qubits: int) -> np.ndarray:
    """Distribution index i = sum_q x_q 2^{n-1-q} (qubit 0 = MSB, reading G4) -> bits."""
    idx = np.asarray(idx, dtype=np.uint64)
    out = np.zeros((idx.shape[0], n_qubits), dtype=np.uint8)
    for q in range(n_qubits):
        out[:, q] = (idx >> np.uint64(n_qubits - 1 - q)) & np.uint64(1)
    return out
