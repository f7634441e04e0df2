"""Pins for oracle/statevector.py and oracle/cutting.py (O1-O5, O7) — CPU only.

Each pin is something other than the oracle itself: closed forms, a brute-force
basis-state loop, the paper's own correctness claim (reconstruction == uncut
distribution, PAPER.md line 195 and Eq. 1), an independent second construction.
"""
import itertools
import os

import numpy as np
import pytest

from oracle import cutting, reconstruct as R, statevector as sv
from tqc_inputs import circuits as C, configs
from tqc_inputs.network import Network

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _golden(name):
    out = {}
    for line in open(os.path.join(GOLDEN, name)):
        if line.strip() and not line.startswith("#"):
            k, *v = line.split()
            out[k] = [float(x) for x in v]
    return out


ALL_GATES = [("y", ()), ("z", ()), ("t", ()), ("tdg", ()), ("cp", (0.9,)), ("h", ()), ("x", ()), ("s", ()), ("sdg", ()), ("sx", ()), ("sy", ()), ("sw", ()),
             ("rx", (0.7,)), ("ry", (1.3,)), ("rz", (2.1,)), ("cz", ()), ("cx", ()), ("rzz", (0.4,))]


@pytest.mark.parametrize("name,params", ALL_GATES)
def test_gates_unitary(name, params):
    u = sv.gate_matrix(name, params)
    assert np.allclose(u @ u.conj().T, np.eye(u.shape[0]), atol=1e-12)


def test_sqrt_gates_square_to_paulis_up_to_phase():
    # sx^2 = -iX etc.: "sqrt(X), sqrt(Y), sqrt(W)" of BASELINE config 1 up to a global phase
    w = (sv.PAULI["X"] + sv.PAULI["Y"]) / np.sqrt(2)
    for nm, p in (("sx", sv.PAULI["X"]), ("sy", sv.PAULI["Y"]), ("sw", w)):
        u = sv.gate_matrix(nm)
        assert np.allclose(u @ u, -1j * p, atol=1e-12)


def test_closed_forms_ghz_h():
    g = _golden("closed_forms.txt")
    p = sv.uncut_probabilities(3, [("h", (), (0,)), ("cx", (), (0, 1)), ("cx", (), (1, 2))])
    assert np.allclose(p, g["ghz3"], atol=1e-12)
    psi = sv.simulate(1, [("h", (), (0,))]).reshape(-1)
    assert np.allclose(psi, [1 / np.sqrt(2)] * 2, atol=1e-12)
    # W-3 -> 1/3 on each one-hot bitstring; W-n and GHZ-n laws of the benchmark generators
    assert np.allclose(sv.uncut_probabilities(3, C.wstate_circuit(3).gates), g["w3"], atol=1e-12)
    for n in (2, 5, 8):
        pw = sv.uncut_probabilities(n, C.wstate_circuit(n).gates)
        hot = [1 << k for k in range(n)]
        assert np.allclose(pw[hot], 1.0 / n, atol=1e-12) and abs(pw.sum() - 1.0) < 1e-12
        pg = sv.uncut_probabilities(n, C.ghz_circuit(n).gates)
        assert np.allclose(pg[[0, 2 ** n - 1]], 0.5, atol=1e-12)


def test_new_gates_against_textbook_identities():
    """y, z, t, tdg, cp are pinned by relations to the already-pinned gates: Y = iXZ, T^2 = S, T Tdg = 1, Z = S^2,
    cp(pi) = cz, cp(l) = phase gates and two cx (the textbook decomposition)."""
    X, S, T = (sv.gate_matrix(nm) for nm in ("x", "s", "t"))
    assert np.allclose(sv.gate_matrix("z"), S @ S) and np.allclose(sv.gate_matrix("y"), 1j * X @ sv.gate_matrix("z"))
    assert np.allclose(T @ T, S) and np.allclose(T @ sv.gate_matrix("tdg"), np.eye(2))
    assert np.allclose(sv.gate_matrix("cp", (np.pi,)), sv.gate_matrix("cz"))
    lam = 0.73
    ph = lambda a: np.diag([1.0, np.exp(1j * a)])
    cx = sv.gate_matrix("cx")
    dec = np.kron(ph(lam / 2), np.eye(2)) @ cx @ np.kron(np.eye(2), ph(-lam / 2)) @ cx @ np.kron(np.eye(2), ph(lam / 2))
    assert np.allclose(dec, sv.gate_matrix("cp", (lam,)), atol=1e-12)


def test_aqft_full_degree_is_the_dft():
    """aqft with no truncation is the quantum Fourier transform without the final swaps: on basis state |x> the output
    amplitudes are those of numpy's DFT read in bit-reversed order (a library routine as the pin)."""
    n = 4
    circ = C.aqft_circuit(n, degree=n)
    for x in (1, 6, 11):
        psi0 = np.zeros((2,) * n, dtype=np.complex128)
        psi0[tuple((x >> (n - 1 - q)) & 1 for q in range(n))] = 1.0
        got = sv.simulate(n, circ.gates, psi0).reshape(-1)
        e = np.zeros(2 ** n); e[x] = 1.0
        want = np.fft.ifft(e) * np.sqrt(2.0 ** n)             # amplitudes exp(+2 pi i x y / N) / sqrt(N)
        rev = [int(format(y, f"0{n}b")[::-1], 2) for y in range(2 ** n)]
        assert np.allclose(got, want[rev], atol=1e-12)


def _brute_force_apply(psi_flat, n, mat, qubits):
    """Textbook definition, basis state by basis state; qubit 0 = MSB; first operand = more significant."""
    out = np.zeros_like(psi_flat)
    k = len(qubits)
    for i in range(2 ** n):
        bits = [(i >> (n - 1 - q)) & 1 for q in range(n)]
        col = 0
        for q in qubits:
            col = col * 2 + bits[q]
        for row in range(2 ** k):
            nb = list(bits)
            for j, q in enumerate(qubits):
                nb[q] = (row >> (k - 1 - j)) & 1
            idx = 0
            for b in nb:
                idx = idx * 2 + b
            out[idx] += mat[row, col] * psi_flat[i]
    return out


@pytest.mark.parametrize("seed", range(4))
def test_simulator_matches_basis_state_loops(seed):
    circ = C.random_small_circuit(4, 6, 100 + seed)
    psi = np.zeros(16, dtype=np.complex128)
    psi[0] = 1
    for (nm, p, qs) in circ.gates:
        psi = _brute_force_apply(psi, 4, sv.gate_matrix(nm, p), qs)
    got = sv.simulate(4, circ.gates).reshape(-1)
    assert np.allclose(got, psi, atol=1e-12)
    assert abs(np.vdot(got, got).real - 1) < 1e-10


def test_cx_orientation():
    # cx controls on its FIRST operand: x on qubit 1 then cx(1, 0) flips qubit 0 -> |11>
    p = sv.uncut_probabilities(2, [("x", (), (1,)), ("cx", (), (1, 0))])
    assert np.allclose(p, [0, 0, 0, 1])


def test_plus_state_pauli_vector_fixture():
    g = _golden("closed_forms.txt")
    sub = cutting.Subcircuit(0, w=1, gates=[("h", (), (0,))], U=[(0, 0)])
    net = Network(1, [(0, 1)], [[0], [0]], [[], [0]])
    assert np.allclose(cutting.build_tensor(net, sub).reshape(-1), g["plus_pauli"], atol=1e-12)
    assert np.allclose(cutting.build_tensor_operator_form(net, sub).reshape(-1), g["plus_pauli"], atol=1e-12)
    # |i> = S H |0> -> (1, 0, 1, 0): pins the sign of the Y setting
    sub.gates = [("h", (), (0,)), ("s", (), (0,))]
    assert np.allclose(cutting.build_tensor(net, sub).reshape(-1), [1, 0, 1, 0], atol=1e-12)


def test_ghz3_through_a_cut():
    g = _golden("closed_forms.txt")
    circ = C.Circuit(3, [("h", (), (0,)), ("cx", (), (0, 1)), ("cx", (), (1, 2))], [None, 0, 1])
    net, T, subs = cutting.tensors_from_circuit(circ)
    assert net.K == 1 and net.m == 2 and net.cuts == [(0, 1)]
    assert [s.w for s in subs] == [2, 2]
    p = R.direct_sum(net, T, R.full_distribution_bits(3))
    assert np.allclose(p, g["ghz3"], atol=1e-12)


def _cut_circuit(n, n2q, m, seed, kmax=6):
    for bump in range(200):
        circ = C.random_small_circuit(n, n2q, seed + 7919 * bump)
        C.assign_parts_random(circ, m, seed + 13 * bump)
        used = sorted(set(p for p in circ.parts if p is not None))
        if used != list(range(m)):
            continue
        net, subs = cutting.extract(circ)
        if 1 <= net.K <= kmax and max(s.w for s in subs) <= 9:
            return circ
    raise AssertionError("no suitable circuit")


@pytest.mark.parametrize("seed", range(12))
def test_reconstruction_equals_uncut_distribution(seed):
    """The paper's correctness claim: P == sum_e (x)_j p_j^e (Eq. 1) — O3..O6 against O7."""
    n = 4 + seed % 4
    circ = _cut_circuit(n, n + 3, 2 + seed % 3, 1000 + seed)
    net, T, subs = cutting.tensors_from_circuit(circ)
    p = R.direct_sum(net, T, R.full_distribution_bits(n))
    truth = sv.uncut_probabilities(n, circ.gates)
    assert np.abs(p - truth).max() <= 1e-8
    assert abs(p.sum() - 1) <= 1e-8 and p.min() >= -1e-8
    # wire budget: sum_s w_s = n + K ; sum_s o_s = n
    assert sum(s.w for s in subs) == n + net.K
    assert sum(net.o(s) for s in range(net.m)) == n
    for s, t in enumerate(T):
        assert abs(t[0].sum() - 2.0 ** net.d(s)) < 1e-9         # sum_x T_s[I..I, x] = 2^{d_s}  (reading G16)
        assert np.abs(t).max() <= 2.0 ** net.d(s) + 1e-9


@pytest.mark.parametrize("seed", range(4))
def test_two_constructions_agree(seed):
    circ = _cut_circuit(5, 8, 2, 2000 + seed, kmax=4)
    net, subs = cutting.extract(circ)
    for sub in subs:
        a = cutting.build_tensor(net, sub)
        b = cutting.build_tensor_operator_form(net, sub)
        assert np.abs(a - b).max() < 1e-12


def test_partition_invariance():
    circ = C.random_small_circuit(6, 9, 31337)
    truth = sv.uncut_probabilities(6, circ.gates)
    results = []
    for pseed in range(40):
        C.assign_parts_random(circ, 2 + pseed % 2, pseed)
        net, subs = cutting.extract(circ)
        if not (1 <= net.K <= 6):
            continue
        T = [cutting.build_tensor(net, s) for s in subs]
        results.append(R.direct_sum(net, T, R.full_distribution_bits(6)))
        if len(results) == 3:
            break
    assert len(results) == 3
    for p in results:
        assert np.abs(p - truth).max() < 1e-8


def test_y_component_present():
    # reading G3: circuits must exercise the Y basis, otherwise a wrong Y sign is invisible
    circ = _cut_circuit(5, 8, 2, 2000, kmax=4)
    net, T, subs = cutting.tensors_from_circuit(circ)
    ymass = 0.0
    for s, t in enumerate(T):
        c = net.c(s)
        t4 = t.reshape((4,) * c + (-1,))
        for ax in range(c):
            ymass += np.abs(np.take(t4, 2, axis=ax)).sum()
    assert ymass > 1e-3


def test_cfg1_shapes_and_reconstruction():
    circ = configs.cfg1_circuit()
    assert sum(1 for g in circ.gates if len(g[2]) == 2) == 9            # (2,2,1,0,2,2) CZs, reading G12
    net, T, subs = cutting.tensors_from_circuit(circ)
    assert (net.m, net.K) == (2, 2) and [s.w for s in subs] == [5, 5]
    assert [t.shape for t in T] == [(16, 16), (16, 16)]
    p = R.direct_sum(net, T, R.full_distribution_bits(8))
    assert np.abs(p - sv.uncut_probabilities(8, circ.gates)).max() < 1e-10


def test_cfg3_shapes():
    net, subs = cutting.extract(configs.cfg3_circuit())
    assert (net.m, net.K) == (3, 6)
    assert [s.w for s in subs] == [12, 12, 12]
    assert [(net.c(s), net.o(s)) for s in range(3)] == [(3, 10), (6, 9), (3, 11)]


def test_cfg2_shapes():
    circ = configs.cfg2_circuit()
    net, subs = cutting.extract(circ)
    assert net.m == 3 and net.K == circ.meta["K"] <= 6
    assert max(s.w for s in subs) <= 10 and sum(s.w for s in subs) == 20 + net.K
