"""O3 subcircuit extraction, O4 variant simulation, O5 Pauli attribution -> T_s, and O5'.

Oracle code (test infrastructure), float64/complex128.  Follows PAPER.md section 2.1
(lines 182-192: upstream cut qubits are measured in {I,X,Y,Z}, I and Z sharing a
setting; downstream cut qubits are initialised in {|0>,|1>,|+>,|i>} and the Pauli bases
are "constructed as a linear combination from the initialization states") and section
6.1.1 (lines 578-594: circuit -> DAG of two-qubit gates, one-qubit gates go with an
adjacent two-qubit gate, terminals are never cut).

The coefficients of the linear combination are NOT in the paper (reading G3); they are
the kappa / sigma tables below, pinned by tests against the uncut statevector (O7), the
independent construction O5' and the |+> fixture (1, 1, 0, 0).
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass, field

import numpy as np

from tqc_inputs.network import Network

from . import statevector as sv

# kappa[k][a]: coefficient of the run prepared in a in (|0>,|1>,|+>,|i>) for downstream basis k in (I,X,Y,Z)
KAPPA = np.array([[1, 1, 0, 0],
                  [-1, -1, 2, 0],
                  [-1, -1, 0, 2],
                  [1, -1, 0, 0]], dtype=np.float64)
_PREP_GATES = {0: (), 1: ("x",), 2: ("h",), 3: ("h", "s")}            # |0>, |1>, |+>, |i>
_MEAS_GATES = {"Z": (), "X": ("h",), "Y": ("sdg", "h")}               # rotate so that Z-measurement reads the basis
_SETTING_OF = ("Z", "X", "Y", "Z")                                       # basis k in (I,X,Y,Z) -> measurement setting
_SIGN = np.array([[1, 1], [1, -1], [1, -1], [1, -1]], dtype=np.float64)  # sigma(k, b)


@dataclass
class Subcircuit:
    sid: int
    w: int = 0
    gates: list = field(default_factory=list)      # (name, params, local wires)
    D: list = field(default_factory=list)          # (local wire, cut id): wire begins at a downstream cut end
    U: list = field(default_factory=list)          # (local wire, cut id): wire ends at an upstream cut end
    O: list = field(default_factory=list)          # (local wire, global qubit): wire ends at a circuit output
    n2q: int = 0


def extract(circ):
    """O3: (Circuit with parts) -> (Network, [Subcircuit])."""
    n, gates, parts = circ.n, circ.gates, circ.parts
    twoq = [[] for _ in range(n)]
    for gi, (_nm, _p, qs) in enumerate(gates):
        if len(qs) == 2:
            assert parts[gi] is not None
            for q in qs:
                twoq[q].append(gi)
    # segments: maximal runs of same-part two-qubit gates on a wire
    segs = []                      # dict(qubit, idx, part, cut_in, cut_out)
    seg_of = {}                    # (gate index, qubit) -> segment id
    wire_segs = [[] for _ in range(n)]
    for q in range(n):
        if not twoq[q]:
            segs.append(dict(qubit=q, idx=0, part=0, cut_in=None, cut_out=None))
            wire_segs[q].append(len(segs) - 1)
            continue
        for gi in twoq[q]:
            if wire_segs[q] and segs[wire_segs[q][-1]]["part"] == parts[gi]:
                sid = wire_segs[q][-1]
            else:
                segs.append(dict(qubit=q, idx=len(wire_segs[q]), part=parts[gi], cut_in=None, cut_out=None))
                sid = len(segs) - 1
                wire_segs[q].append(sid)
            seg_of[(gi, q)] = sid
    # one-qubit gates: nearest preceding two-qubit gate on the wire, else the following one
    for gi, (_nm, _p, qs) in enumerate(gates):
        if len(qs) == 1:
            q = qs[0]
            before = [g for g in twoq[q] if g < gi]
            if before:
                seg_of[(gi, q)] = seg_of[(before[-1], q)]
            elif twoq[q]:
                seg_of[(gi, q)] = seg_of[(twoq[q][0], q)]
            else:
                seg_of[(gi, q)] = wire_segs[q][0]
    # cuts: between consecutive segments of a wire; upstream = earlier
    cuts = []
    for q in range(n):
        for a, b in zip(wire_segs[q][:-1], wire_segs[q][1:]):
            e = len(cuts)
            cuts.append((segs[a]["part"], segs[b]["part"]))
            segs[a]["cut_out"] = e
            segs[b]["cut_in"] = e
    m = max(s["part"] for s in segs) + 1
    subs = [Subcircuit(s) for s in range(m)]
    local = {}
    for sid in sorted(range(len(segs)), key=lambda i: (segs[i]["part"], segs[i]["qubit"], segs[i]["idx"])):
        s = segs[sid]
        sub = subs[s["part"]]
        local[sid] = sub.w
        if s["cut_in"] is not None:
            sub.D.append((sub.w, s["cut_in"]))
        if s["cut_out"] is not None:
            sub.U.append((sub.w, s["cut_out"]))
        else:
            sub.O.append((sub.w, s["qubit"]))
        sub.w += 1
    for gi, (nm, p, qs) in enumerate(gates):
        sids = [seg_of[(gi, q)] for q in qs]
        part = segs[sids[0]]["part"]
        assert all(segs[x]["part"] == part for x in sids)
        subs[part].gates.append((nm, p, tuple(local[x] for x in sids)))
        subs[part].n2q += len(qs) == 2
    sub_cuts = [sorted([e for (_w, e) in sub.D] + [e for (_w, e) in sub.U]) for sub in subs]
    sub_qubits = [[q for (_w, q) in sub.O] for sub in subs]
    net = Network(n, cuts, sub_cuts, sub_qubits, name=circ.name,
                  meta={"w": [sub.w for sub in subs], "n2q": [sub.n2q for sub in subs]})
    net.validate()
    return net, subs


def _run(sub: Subcircuit, prep_gates_per_D):
    psi = sv.zero_state(sub.w)
    for (wire, _e), names in zip(sub.D, prep_gates_per_D):
        for nm in names:
            psi = sv.apply_gate(psi, sv.gate_matrix(nm), (wire,))
    return sv.simulate(sub.w, sub.gates, psi)


def build_tensor(net: Network, sub: Subcircuit) -> np.ndarray:
    """O4 + O5: T_s as [4^{c_s}][2^{o_s}] float64, bond axes in net.sub_cuts[s] order."""
    d, u, o = len(sub.D), len(sub.U), len(sub.O)
    u_wires = [w for (w, _e) in sub.U]
    R = np.zeros((4,) * d + (4,) * u + (2 ** o,), dtype=np.float64)
    for a in itertools.product(range(4), repeat=d):                      # 4^d preparations
        psi = _run(sub, [_PREP_GATES[ai] for ai in a])
        probs = {}
        for beta in itertools.product("ZXY", repeat=u):                  # 3^u measurement settings
            phi = psi
            for wire, b in zip(u_wires, beta):
                for nm in _MEAS_GATES[b]:
                    phi = sv.apply_gate(phi, sv.gate_matrix(nm), (wire,))
            probs[beta] = phi.real ** 2 + phi.imag ** 2
        for ku in itertools.product(range(4), repeat=u):
            q = probs[tuple(_SETTING_OF[k] for k in ku)]
            # sum over measured bits b_U with signs sigma(k, b); contract highest axis first
            for wire, k in sorted(zip(u_wires, ku), reverse=True):
                q = np.tensordot(q, _SIGN[k], axes=([wire], [0]))
            R[a + ku] = q.reshape(-1)
    for i in range(d):                                                   # downstream linear combination
        R = np.moveaxis(np.tensordot(KAPPA, R, axes=([1], [i])), 0, i)
    return _order_axes(net, sub, R)


def _order_axes(net, sub, R):
    have = [e for (_w, e) in sub.D] + [e for (_w, e) in sub.U]
    want = net.sub_cuts[sub.sid]
    perm = [have.index(e) for e in want] + [len(have)]
    c, o = len(have), len(sub.O)
    return np.ascontiguousarray(np.transpose(R, perm)).reshape(4 ** c, 2 ** o)


_EIG_PREP = {0: ((("",), 1.0), (("x",), 1.0)),          # I = |0><0| + |1><1|
             1: ((("h",), 1.0), (("x", "h"), -1.0)),    # X = |+><+| - |-><-|
             2: ((("h", "s"), 1.0), (("h", "sdg"), -1.0)),  # Y = |i><i| - |-i><-i|
             3: ((("",), 1.0), (("x",), -1.0))}         # Z = |0><0| - |1><1|


def build_tensor_operator_form(net: Network, sub: Subcircuit) -> np.ndarray:
    """O5': T_s[k_d, k_u, x] = Tr[(|x><x|_O (x) P_{k_u}) C ( (x)_i P_{k_d,i} (x) |0><0| ) C^dagger]
    with each downstream Pauli written in its own eigenbasis and each upstream Pauli applied
    as an operator to the amplitudes — no measurement rotations, no kappa table."""
    d, u, o = len(sub.D), len(sub.U), len(sub.O)
    u_wires = [w for (w, _e) in sub.U]
    paulis = [sv.PAULI[c] for c in "IXYZ"]
    R = np.zeros((4,) * d + (4,) * u + (2 ** o,), dtype=np.float64)
    for kd in itertools.product(range(4), repeat=d):
        for choice in itertools.product(range(2), repeat=d):
            sign = 1.0
            preps = []
            for k, ch in zip(kd, choice):
                names, s = _EIG_PREP[k][ch]
                preps.append(tuple(nm for nm in names if nm))
                sign *= s
            psi = _run(sub, preps)
            for ku in itertools.product(range(4), repeat=u):
                phi = psi
                for wire, k in zip(u_wires, ku):
                    phi = sv.apply_gate(phi, paulis[k], (wire,))
                val = (np.conj(psi) * phi).real
                for wire in sorted(u_wires, reverse=True):
                    val = val.sum(axis=wire)
                R[kd + ku] += sign * val.reshape(-1)
    return _order_axes(net, sub, R)


def tensors_from_circuit(circ, operator_form: bool = False):
    """(Network, [T_s float64]) for a circuit with a gate->subcircuit assignment."""
    net, subs = extract(circ)
    build = build_tensor_operator_form if operator_form else build_tensor
    return net, [build(net, sub) for sub in subs], subs
