"""O1 gates, O2 dense statevector simulation, O7 uncut reference probabilities.

Oracle code (test infrastructure): float64/complex128, plain numpy.
The paper uses "noiseless classical simulators" as the stand-in for QPUs
(PAPER.md line 722); this is such a simulator.  Bit convention (reading G4,
S:81): qubit 0 is the most significant bit of a state index, i.e. axis 0 of the
(2,)*w amplitude tensor.
"""
from __future__ import annotations

import numpy as np

_I2 = np.eye(2, dtype=np.complex128)
_X = np.array([[0, 1], [1, 0]], dtype=np.complex128)
_Y = np.array([[0, -1j], [1j, 0]], dtype=np.complex128)
_Z = np.array([[1, 0], [0, -1]], dtype=np.complex128)
_W = (_X + _Y) / np.sqrt(2.0)
PAULI = {"I": _I2, "X": _X, "Y": _Y, "Z": _Z}


def gate_matrix(name: str, params=()) -> np.ndarray:
    """Standard definitions (O1).  sx/sy/sw = exp(-i pi/4 P) = (I - iP)/sqrt2 for
    P = X, Y, W = (X+Y)/sqrt2: sqrt(X), sqrt(Y), sqrt(W) up to a global phase (reading G11).
    Two-qubit matrices act on (first operand, second operand) with the first as the
    more significant bit; cx controls on its first operand."""
    if name == "h":
        return np.array([[1, 1], [1, -1]], dtype=np.complex128) / np.sqrt(2.0)
    if name == "x":
        return _X.copy()
    if name == "y":
        return _Y.copy()
    if name == "z":
        return _Z.copy()
    if name == "t":
        return np.array([[1, 0], [0, np.exp(0.25j * np.pi)]], dtype=np.complex128)
    if name == "tdg":
        return np.array([[1, 0], [0, np.exp(-0.25j * np.pi)]], dtype=np.complex128)
    if name == "s":
        return np.array([[1, 0], [0, 1j]], dtype=np.complex128)
    if name == "sdg":
        return np.array([[1, 0], [0, -1j]], dtype=np.complex128)
    if name in ("sx", "sy", "sw"):
        p = {"sx": _X, "sy": _Y, "sw": _W}[name]
        return (_I2 - 1j * p) / np.sqrt(2.0)
    if name in ("rx", "ry", "rz"):
        (theta,) = params
        p = {"rx": _X, "ry": _Y, "rz": _Z}[name]
        return np.cos(theta / 2.0) * _I2 - 1j * np.sin(theta / 2.0) * p
    if name == "cz":
        return np.diag([1, 1, 1, -1]).astype(np.complex128)
    if name == "cx":
        return np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 0, 1], [0, 0, 1, 0]], dtype=np.complex128)
    if name == "cp":                                           # controlled phase: |11> picks up e^{i lambda}
        (lam,) = params
        return np.diag([1, 1, 1, np.exp(1j * lam)]).astype(np.complex128)
    if name == "rzz":
        (gamma,) = params
        return np.diag(np.exp(-1j * gamma * np.array([1, -1, -1, 1]))).astype(np.complex128)
    raise ValueError(f"unknown gate {name}")


def zero_state(w: int) -> np.ndarray:
    psi = np.zeros((2,) * w, dtype=np.complex128)
    psi[(0,) * w] = 1.0
    return psi


def apply_gate(psi: np.ndarray, mat: np.ndarray, qubits) -> np.ndarray:
    """psi'[..a'..b'..] = sum_{a,b} U[(a',b'),(a,b)] psi[..a..b..]."""
    k = len(qubits)
    u = mat.reshape((2,) * (2 * k))
    out = np.tensordot(u, psi, axes=(list(range(k, 2 * k)), list(qubits)))
    # tensordot puts the new axes first; move them back to the operand positions
    return np.moveaxis(out, list(range(k)), list(qubits))


def simulate(n: int, gates, psi0: np.ndarray | None = None) -> np.ndarray:
    """Apply gates in program order to |0...0> (or psi0); returns the (2,)*n amplitude tensor."""
    psi = zero_state(n) if psi0 is None else psi0
    for (name, params, qubits) in gates:
        psi = apply_gate(psi, gate_matrix(name, params), qubits)
    return psi


def uncut_probabilities(n: int, gates) -> np.ndarray:
    """O7: p_true(x) = |amp_x|^2 as a flat vector, index = sum_q x_q 2^{n-1-q}."""
    psi = simulate(n, gates)
    return (psi.real ** 2 + psi.imag ** 2).reshape(-1)
