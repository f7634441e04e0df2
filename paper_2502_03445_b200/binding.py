"""ctypes binding of libtqc.so (include/tqc.h).  Argument marshalling only.

The four entry points carry the C names: tqc_plan, tqc_load_subcircuit_tensors,
tqc_contract_states, tqc_contract_distribution.  Device buffers are torch tensors whose
data_ptr() is passed through; the stream is torch's current CUDA stream.  There is no CPU
fallback: if libtqc.so has not been built the import raises, and a compute call without a
CUDA device raises TqcError(TQC_E_CUDA).
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_char_p, c_double, c_int, c_int32, c_int64, c_size_t, c_uint64, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libtqc.so")

MODE_STATES, MODE_DISTRIBUTION = 0, 1
KERNEL_SIMT_TILE, KERNEL_DOT, KERNEL_TCGEN05 = 0, 1, 2
NODE_LEAF, NODE_TABLE, NODE_BATCH = 0, 1, 2

STATUS_NAMES = {0: "TQC_OK", -1: "TQC_E_ARG", -2: "TQC_E_SHAPE", -3: "TQC_E_STATE", -4: "TQC_E_INFEASIBLE",
                -5: "TQC_E_WORKSPACE", -6: "TQC_E_TOO_LARGE", -7: "TQC_E_CUDA", -8: "TQC_E_PARSE"}

# every symbol include/tqc.h declares (tests check that the library exports each one)
EXPORTED = ["tqc_plan", "tqc_plan_destroy", "tqc_plan_mode", "tqc_plan_num_qubits", "tqc_plan_num_subcircuits",
            "tqc_plan_num_cuts", "tqc_plan_num_steps", "tqc_plan_kmax", "tqc_plan_tensor_shape", "tqc_plan_step",
            "tqc_plan_node", "tqc_plan_cost_log2", "tqc_plan_serialize", "tqc_plan_workspace_bytes",
            "tqc_plan_workspace_min_bytes", "tqc_load_subcircuit_tensors", "tqc_contract_states",
            "tqc_contract_distribution", "tqc_plan_launch_count", "tqc_last_error", "tqc_version",
            "tqc_plan_workspace_bytes_host", "tqc_contract_states_host", "tqc_contract_distribution_host",
            "tqc_plan_profile_enable", "tqc_plan_profile_read", "tqc_plan_chain_status", "tqc_hss_scores", "tqc_hss_select",
            "tqc_hss_expand", "tqc_plan_num_sliced_cuts", "tqc_choose_slice_cuts", "tqc_hss_prepare",
            "tqc_hss_workspace_bytes", "tqc_hss_cost_log2", "tqc_hss_contract", "tqc_simulate_workspace_bytes",
            "tqc_simulate_subcircuit_tensor", "tqc_simulate_subcircuit_tensor_static", "tqc_static_scratch_bytes",
            "tqc_plan_finalize", "tqc_plan_from_circuit", "tqc_plan_from_gates",
            "tqc_plan_cut_network", "tqc_plan_cut_subcircuit", "tqc_plan_cut_assignment", "tqc_cut_merging_cost",
            "tqc_plan_cost_report", "tqc_plan_pair_launch_count", "tqc_plan_modelled_seconds_per_state"]


class TqcError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{STATUS_NAMES.get(code, code)}: {msg}")
        self.code = code


class _NetworkDesc(ctypes.Structure):
    _fields_ = [("n_qubits", c_int32), ("m", c_int32), ("K", c_int32),
                ("cut_up", POINTER(c_int32)), ("cut_down", POINTER(c_int32)),
                ("sub_cut_ofs", POINTER(c_int32)), ("sub_cuts", POINTER(c_int32)),
                ("sub_qubit_ofs", POINTER(c_int32)), ("sub_qubits", POINTER(c_int32))]


class _PlanOpts(ctypes.Structure):
    _fields_ = [("mode", c_int32), ("n_order_steps", c_int32), ("order", POINTER(c_int32)),
                ("restarts", c_int32), ("seed", c_uint64), ("batch_hint", c_int64),
                ("table_log2_floats_max", c_int32), ("use_tcgen05", c_int32), ("use_chain", c_int32),
                ("n_slice_cuts", c_int32), ("slice_cuts", POINTER(c_int32)), ("kmax_cap", c_int32), ("objective", c_int32)]


class _Gate(ctypes.Structure):
    _fields_ = [("kind", c_int32), ("wire0", c_int32), ("wire1", c_int32), ("reserved", c_int32), ("param", c_double)]


class _SubcircuitDesc(ctypes.Structure):
    _fields_ = [("w", c_int32), ("n_gates", c_int32), ("gates", POINTER(_Gate)),
                ("d", c_int32), ("u", c_int32), ("o", c_int32), ("fuse_gates", c_int32),
                ("D_wires", POINTER(c_int32)), ("U_wires", POINTER(c_int32)), ("O_wires", POINTER(c_int32)),
                ("bond_pos", POINTER(c_int32)), ("walk_settings", c_int32), ("reserved", c_int32)]


class _CutOpts(ctypes.Structure):
    _fields_ = [("w_max", c_int32), ("s_max", c_int32), ("K_t", c_int32), ("reserved", c_int32), ("Q_max", c_double)]


class _CostModel(ctypes.Structure):
    _fields_ = [("t_g", c_double), ("t_m", c_double), ("flops", c_double), ("n_qpus", c_int32),
                ("shots_log2_min", c_int32), ("shots_log2_max", c_int32), ("reserved", c_int32)]


class _CostReport(ctypes.Structure):
    _fields_ = [("t_qpu", c_double), ("t_classical", c_double), ("t_total", c_double), ("c_tn_flop", c_double),
                ("qpu_variants", c_double)]


GATE_KINDS = {"h": 0, "x": 1, "s": 2, "sdg": 3, "sx": 4, "sy": 5, "sw": 6, "rx": 7, "ry": 8, "rz": 9, "cz": 10, "cx": 11,
              "rzz": 12, "y": 13, "z": 14, "t": 15, "tdg": 16, "cp": 17}
GATE_NAMES = {v: k for k, v in GATE_KINDS.items()}


def lib_path() -> str:
    return _LIB_PATH


def _load() -> ctypes.CDLL:
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_2502_03445_b200.build` "
                          "(there is no CPU fallback)")
    lib = ctypes.CDLL(_LIB_PATH)
    lib.tqc_last_error.restype = c_char_p
    lib.tqc_version.restype = c_char_p
    lib.tqc_plan.argtypes = [POINTER(_NetworkDesc), POINTER(_PlanOpts), POINTER(c_void_p)]
    lib.tqc_choose_slice_cuts.argtypes = [POINTER(_NetworkDesc), POINTER(_PlanOpts), c_int, c_int, c_void_p, POINTER(c_int32)]
    lib.tqc_plan_destroy.argtypes = [c_void_p]
    lib.tqc_plan_destroy.restype = None
    for name in ("tqc_plan_mode", "tqc_plan_num_qubits", "tqc_plan_num_subcircuits", "tqc_plan_num_cuts",
                 "tqc_plan_num_steps", "tqc_plan_kmax", "tqc_plan_num_sliced_cuts"):
        getattr(lib, name).argtypes = [c_void_p]
    lib.tqc_plan_tensor_shape.argtypes = [c_void_p, c_int, POINTER(c_int), POINTER(c_int)]
    lib.tqc_plan_step.argtypes = [c_void_p, c_int] + [POINTER(c_int)] * 7
    lib.tqc_plan_node.argtypes = [c_void_p, c_int] + [POINTER(c_int)] * 3
    lib.tqc_plan_cost_log2.argtypes = [c_void_p]
    lib.tqc_plan_cost_log2.restype = c_double
    lib.tqc_plan_modelled_seconds_per_state.argtypes = [c_void_p]
    lib.tqc_plan_modelled_seconds_per_state.restype = c_double
    lib.tqc_plan_serialize.argtypes = [c_void_p, c_void_p, POINTER(c_size_t)]
    lib.tqc_plan_workspace_bytes.argtypes = [c_void_p, c_size_t, c_int]
    lib.tqc_plan_workspace_bytes.restype = c_size_t
    lib.tqc_plan_workspace_min_bytes.argtypes = [c_void_p]
    lib.tqc_plan_workspace_min_bytes.restype = c_size_t
    lib.tqc_load_subcircuit_tensors.argtypes = [c_void_p, c_int, c_void_p, c_size_t, c_int, c_void_p]
    lib.tqc_plan_finalize.argtypes = [c_void_p, c_void_p]
    lib.tqc_contract_states.argtypes = [c_void_p, c_void_p, c_size_t, c_void_p, c_void_p, c_size_t, c_void_p]
    lib.tqc_contract_distribution.argtypes = [c_void_p, c_uint64, c_int, c_void_p, c_void_p, c_size_t, c_void_p]
    lib.tqc_plan_launch_count.argtypes = [c_void_p]
    lib.tqc_plan_launch_count.restype = c_uint64
    lib.tqc_plan_pair_launch_count.argtypes = [c_void_p]
    lib.tqc_plan_pair_launch_count.restype = c_uint64
    lib.tqc_plan_workspace_bytes_host.argtypes = [c_void_p, c_size_t, c_int]
    lib.tqc_plan_workspace_bytes_host.restype = c_size_t
    lib.tqc_contract_states_host.argtypes = [c_void_p, c_void_p, c_size_t, c_void_p, c_void_p, c_size_t, c_void_p]
    lib.tqc_contract_distribution_host.argtypes = [c_void_p, c_uint64, c_int, c_void_p, c_void_p, c_size_t, c_void_p]
    lib.tqc_plan_chain_status.argtypes = [c_void_p, c_char_p, c_size_t]
    lib.tqc_plan_profile_enable.argtypes = [c_void_p, c_int]
    lib.tqc_plan_profile_read.argtypes = [c_void_p, c_void_p, c_void_p, POINTER(c_size_t)]
    lib.tqc_hss_scores.argtypes = [c_void_p, c_int, c_void_p, c_void_p]
    lib.tqc_hss_select.argtypes = [c_void_p, POINTER(c_void_p), c_uint64, c_void_p, c_void_p, c_size_t]
    lib.tqc_hss_expand.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_size_t, POINTER(c_size_t)]
    lib.tqc_hss_prepare.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p]
    lib.tqc_hss_workspace_bytes.argtypes = [c_void_p]
    lib.tqc_hss_workspace_bytes.restype = c_size_t
    lib.tqc_hss_cost_log2.argtypes = [c_void_p]
    lib.tqc_hss_cost_log2.restype = c_double
    lib.tqc_hss_contract.argtypes = [c_void_p, c_void_p, c_void_p, c_size_t, c_void_p]
    lib.tqc_simulate_workspace_bytes.argtypes = [POINTER(_SubcircuitDesc)]
    lib.tqc_simulate_workspace_bytes.restype = c_size_t
    lib.tqc_simulate_subcircuit_tensor.argtypes = [POINTER(_SubcircuitDesc), c_void_p, c_void_p, c_size_t, c_void_p]
    lib.tqc_simulate_subcircuit_tensor_static.argtypes = [POINTER(_SubcircuitDesc), c_void_p, c_void_p]
    lib.tqc_static_scratch_bytes.argtypes = []
    lib.tqc_static_scratch_bytes.restype = c_size_t
    lib.tqc_plan_from_circuit.argtypes = [c_char_p, POINTER(_CutOpts), POINTER(_PlanOpts), POINTER(c_void_p)]
    lib.tqc_plan_from_gates.argtypes = [c_int, POINTER(_Gate), c_int, POINTER(_CutOpts), POINTER(_PlanOpts), POINTER(c_void_p)]
    lib.tqc_plan_cut_network.argtypes = [c_void_p, POINTER(_NetworkDesc)]
    lib.tqc_plan_cut_subcircuit.argtypes = [c_void_p, c_int, POINTER(_SubcircuitDesc), POINTER(c_int32), POINTER(c_int32)]
    lib.tqc_plan_cut_assignment.argtypes = [c_void_p, c_void_p, c_size_t]
    lib.tqc_cut_merging_cost.argtypes = [c_int] * 6
    lib.tqc_cut_merging_cost.restype = c_double
    lib.tqc_plan_cost_report.argtypes = [c_void_p, POINTER(_CostModel), c_void_p, c_double, POINTER(_CostReport)]
    return lib


_lib = _load()


def _check(rc: int) -> None:
    if rc != 0:
        raise TqcError(rc, _lib.tqc_last_error().decode())


def version() -> str:
    return _lib.tqc_version().decode()


def _i32(values):
    arr = np.ascontiguousarray(np.asarray(list(values), dtype=np.int32))
    if arr.size == 0:
        arr = np.zeros(1, dtype=np.int32)
    return arr, arr.ctypes.data_as(POINTER(c_int32))


def _stream_ptr(stream) -> int:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


class Plan:
    """Owner of a tqc_plan_t handle (plan + the library's device copies of the tensors)."""

    def __init__(self, handle: int):
        self._h = c_void_p(handle)

    def close(self) -> None:
        if self._h:
            _lib.tqc_plan_destroy(self._h)
            self._h = c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- queries --------------------------------------------------------------------------
    @property
    def mode(self) -> int: return _lib.tqc_plan_mode(self._h)
    @property
    def n_qubits(self) -> int: return _lib.tqc_plan_num_qubits(self._h)
    @property
    def m(self) -> int: return _lib.tqc_plan_num_subcircuits(self._h)
    @property
    def K(self) -> int: return _lib.tqc_plan_num_cuts(self._h)
    @property
    def n_sliced_cuts(self) -> int: return _lib.tqc_plan_num_sliced_cuts(self._h)
    @property
    def num_steps(self) -> int: return _lib.tqc_plan_num_steps(self._h)
    @property
    def kmax(self) -> int: return _lib.tqc_plan_kmax(self._h)
    @property
    def cost_log2(self) -> float: return _lib.tqc_plan_cost_log2(self._h)
    @property
    def modelled_seconds_per_state(self) -> float: return _lib.tqc_plan_modelled_seconds_per_state(self._h)
    @property
    def launch_count(self) -> int: return int(_lib.tqc_plan_launch_count(self._h))
    @property
    def pair_launch_count(self) -> int: return int(_lib.tqc_plan_pair_launch_count(self._h))

    def tensor_shape(self, s: int):
        c, o = c_int(), c_int()
        _check(_lib.tqc_plan_tensor_shape(self._h, s, byref(c), byref(o)))
        return c.value, o.value

    def step(self, i: int) -> dict:
        v = [c_int() for _ in range(7)]
        _check(_lib.tqc_plan_step(self._h, i, *[byref(x) for x in v]))
        names = ("lhs", "rhs", "n_inner", "n_outer_lhs", "n_outer_rhs", "log2cost", "kernel_class")
        return {k: x.value for k, x in zip(names, v)}

    def node(self, v: int) -> dict:
        out = [c_int() for _ in range(3)]
        _check(_lib.tqc_plan_node(self._h, v, *[byref(x) for x in out]))
        return {k: x.value for k, x in zip(("kind", "n_bits", "n_open"), out)}

    def steps(self):
        return [self.step(i) for i in range(self.num_steps)]

    def serialize(self) -> bytes:
        n = c_size_t(0)
        _check(_lib.tqc_plan_serialize(self._h, None, byref(n)))
        buf = ctypes.create_string_buffer(n.value)
        _check(_lib.tqc_plan_serialize(self._h, buf, byref(n)))
        return buf.raw[:n.value]

    def workspace_bytes(self, n_states: int = 0, prefix_bits: int = 0) -> int:
        return int(_lib.tqc_plan_workspace_bytes(self._h, n_states, prefix_bits))

    def workspace_min_bytes(self) -> int:
        return int(_lib.tqc_plan_workspace_min_bytes(self._h))

    def workspace_bytes_host(self, n_states: int = 0, prefix_bits: int = 0) -> int:
        return int(_lib.tqc_plan_workspace_bytes_host(self._h, n_states, prefix_bits))

    # ---- plans made from a circuit (tqc_plan_from_circuit / tqc_plan_from_gates) ----------------
    def cut_network(self):
        """The cut network the partitioner produced: an object with n_qubits, cuts [(up, down)], sub_cuts, sub_qubits
        (the attributes tqc_plan reads), plus m and K."""
        from types import SimpleNamespace
        d = _NetworkDesc()
        _check(_lib.tqc_plan_cut_network(self._h, byref(d)))
        cuts = [(int(d.cut_up[e]), int(d.cut_down[e])) for e in range(d.K)]
        sub_cuts = [[int(d.sub_cuts[j]) for j in range(d.sub_cut_ofs[s], d.sub_cut_ofs[s + 1])] for s in range(d.m)]
        sub_qubits = [[int(d.sub_qubits[j]) for j in range(d.sub_qubit_ofs[s], d.sub_qubit_ofs[s + 1])] for s in range(d.m)]
        return SimpleNamespace(n_qubits=int(d.n_qubits), m=int(d.m), K=int(d.K), cuts=cuts, sub_cuts=sub_cuts,
                               sub_qubits=sub_qubits)

    def cut_subcircuit(self, s: int) -> dict:
        """Subcircuit s in the argument form of tqc_simulate_subcircuit_tensor (w, gates, D_wires, U_wires, O_wires,
        bond_pos) plus n2q (two-qubit gates) and depth (t_s)."""
        d = _SubcircuitDesc()
        n2q, depth = c_int32(), c_int32()
        _check(_lib.tqc_plan_cut_subcircuit(self._h, s, byref(d), byref(n2q), byref(depth)))
        gates = []
        for t in range(d.n_gates):
            g = d.gates[t]
            name = GATE_NAMES[int(g.kind)]
            two = name in ("cz", "cx", "rzz", "cp")
            has_param = name in ("rx", "ry", "rz", "rzz", "cp")
            gates.append((name, (float(g.param),) if has_param else (), (int(g.wire0), int(g.wire1)) if two else (int(g.wire0),)))
        return dict(w=int(d.w), gates=gates, D_wires=[int(d.D_wires[i]) for i in range(d.d)],
                    U_wires=[int(d.U_wires[i]) for i in range(d.u)], O_wires=[int(d.O_wires[i]) for i in range(d.o)],
                    bond_pos=[int(d.bond_pos[i]) for i in range(d.d + d.u)], n2q=int(n2q.value), depth=int(depth.value))

    def cut_assignment(self, n_gates: int):
        out = np.zeros(max(1, n_gates), dtype=np.int32)
        _check(_lib.tqc_plan_cut_assignment(self._h, out.ctypes.data, n_gates))
        return [int(x) for x in out[:n_gates]]

    def cost_report(self, flops: float, n_states: float = 1.0, depth=None, t_g: float = 0.0, t_m: float = 0.0,
                    n_qpus: int = 0, shots_log2_min: int = 0, shots_log2_max: int = 0) -> dict:
        """Eqs. 4-6 of the paper for this plan (include/tqc.h)."""
        model = _CostModel(t_g, t_m, flops, n_qpus, shots_log2_min, shots_log2_max, 0)
        rep = _CostReport()
        darr = None if depth is None else np.ascontiguousarray(np.asarray(depth, dtype=np.int32))
        _check(_lib.tqc_plan_cost_report(self._h, byref(model), None if darr is None else darr.ctypes.data, float(n_states),
                                         byref(rep)))
        return {k: float(getattr(rep, k)) for k in ("t_qpu", "t_classical", "t_total", "c_tn_flop", "qpu_variants")}

    def finalize(self, stream=None) -> None:
        """tqc_plan_finalize: device tables, specialised chain kernel, side streams (implicit at the last tensor load)."""
        _check(_lib.tqc_plan_finalize(self._h, _stream_ptr(stream)))

    def chain_status(self):
        """(0 no fused chain | 1 generic chain kernel | 2 plan-specialised chain kernel, note)."""
        buf = ctypes.create_string_buffer(4096)
        rc = _lib.tqc_plan_chain_status(self._h, buf, 4096)
        return rc, buf.value.decode(errors="replace")

    @property
    def hss_cost_log2(self) -> float:
        """log2 multiplications of the pruned contraction planned by the last tqc_hss_prepare / tqc_hss_contract (< 0: none)."""
        return float(_lib.tqc_hss_cost_log2(self._h))

    def profile_enable(self, on: bool = True) -> None:
        _check(_lib.tqc_plan_profile_enable(self._h, 1 if on else 0))

    def profile_read(self):
        """[(tag, ms)] per launch of the last profiled contract call (waits for it)."""
        n = c_size_t(0)
        _check(_lib.tqc_plan_profile_read(self._h, None, None, byref(n)))
        tags = np.zeros(max(1, n.value), dtype=np.int32)
        ms = np.zeros(max(1, n.value), dtype=np.float32)
        _check(_lib.tqc_plan_profile_read(self._h, tags.ctypes.data, ms.ctypes.data, byref(n)))
        return [(int(tags[i]), float(ms[i])) for i in range(n.value)]


def _network_desc(net):
    m = len(net.sub_cuts)
    keep = [_i32(c[0] for c in net.cuts), _i32(c[1] for c in net.cuts),
            _i32(np.concatenate([[0], np.cumsum([len(x) for x in net.sub_cuts])])), _i32(e for x in net.sub_cuts for e in x),
            _i32(np.concatenate([[0], np.cumsum([len(x) for x in net.sub_qubits])])), _i32(q for x in net.sub_qubits for q in x)]
    desc = _NetworkDesc(net.n_qubits, m, len(net.cuts), *[k[1] for k in keep])
    return desc, keep                      # keep: the arrays the descriptor points into


def tqc_plan(net, mode: int = MODE_STATES, order=None, restarts: int = 0, seed: int = 0, batch_hint: int = 0,
             table_log2_floats_max: int = 0, use_tcgen05: int = 0, use_chain: int = 0, slice_cuts=None,
             kmax_cap: int = 0, objective: int = 0) -> Plan:
    """net: any object with n_qubits, cuts [(up, down)], sub_cuts [[cut ids]], sub_qubits [[qubit ids]]
    (e.g. tqc_inputs.Network).  order: optional list of m-1 (lhs, rhs) node-id pairs.  slice_cuts: cut ids evaluated by
    index slicing (summed over their 4 bases) instead of being contracted as bonds."""
    desc, _keep = _network_desc(net)
    oflat, oflat_p = _i32(v for ab in (order or []) for v in ab)
    sflat, sflat_p = _i32(slice_cuts or [])
    opts = _PlanOpts(mode, len(order) if order else 0, oflat_p, restarts, seed, batch_hint,
                     table_log2_floats_max, use_tcgen05, use_chain, len(slice_cuts) if slice_cuts else 0, sflat_p,
                     kmax_cap, objective)
    h = c_void_p()
    _check(_lib.tqc_plan(byref(desc), byref(opts), byref(h)))
    return Plan(h.value)


def _gate_array(gates):
    garr = (_Gate * max(1, len(gates)))()
    for t, (name, params, wires) in enumerate(gates):
        if name not in GATE_KINDS:
            raise TqcError(-1, f"unknown gate {name}")
        garr[t].kind = GATE_KINDS[name]
        garr[t].wire0 = int(wires[0])
        garr[t].wire1 = int(wires[1]) if len(wires) > 1 else 0
        garr[t].param = float(params[0]) if len(params) else 0.0
    return garr


def circuit_text(n_qubits: int, gates) -> str:
    """The circuit text tqc_plan_from_circuit parses: `qubits n`, then `<name>[(<angle>)] q0 [q1]` per gate."""
    lines = [f"qubits {n_qubits}"]
    for (name, params, wires) in gates:
        arg = f"({float(params[0])!r})" if len(params) else ""
        lines.append(f"{name}{arg} " + " ".join(str(int(q)) for q in wires))
    return "\n".join(lines) + "\n"


def _plan_opts_simple(mode, restarts, seed, batch_hint, table_log2_floats_max, use_tcgen05, use_chain, kmax_cap):
    return _PlanOpts(mode, 0, None, restarts, seed, batch_hint, table_log2_floats_max, use_tcgen05, use_chain, 0, None, kmax_cap, 0)


def tqc_plan_from_circuit(text: str, w_max: int, s_max: int, K_t: int = 0, Q_max: float = 0.0, mode: int = MODE_STATES,
                          restarts: int = 0, seed: int = 0, batch_hint: int = 0, table_log2_floats_max: int = 0,
                          use_tcgen05: int = 0, use_chain: int = 0, kmax_cap: int = 0) -> Plan:
    """Circuit text -> DAG -> Greedy Graph Growing partition under (w_max, s_max) -> cut network -> plan (section 6)."""
    cut = _CutOpts(w_max, s_max, K_t, 0, Q_max)
    opts = _plan_opts_simple(mode, restarts, seed, batch_hint, table_log2_floats_max, use_tcgen05, use_chain, kmax_cap)
    h = c_void_p()
    _check(_lib.tqc_plan_from_circuit(text.encode(), byref(cut), byref(opts), byref(h)))
    return Plan(h.value)


def tqc_plan_from_gates(n_qubits: int, gates, w_max: int, s_max: int, K_t: int = 0, Q_max: float = 0.0,
                        mode: int = MODE_STATES, restarts: int = 0, seed: int = 0, batch_hint: int = 0,
                        table_log2_floats_max: int = 0, use_tcgen05: int = 0, use_chain: int = 0, kmax_cap: int = 0) -> Plan:
    """The same from a gate list [(name, params, qubits)]."""
    garr = _gate_array(gates)
    cut = _CutOpts(w_max, s_max, K_t, 0, Q_max)
    opts = _plan_opts_simple(mode, restarts, seed, batch_hint, table_log2_floats_max, use_tcgen05, use_chain, kmax_cap)
    h = c_void_p()
    _check(_lib.tqc_plan_from_gates(n_qubits, garr, len(gates), byref(cut), byref(opts), byref(h)))
    return Plan(h.value)


def tqc_cut_merging_cost(w_trial: int, w_max: int, s_trial: int, s_max: int, K_trial: int, K_t: int) -> float:
    """Table 1 of the paper; negative = not allowed."""
    return float(_lib.tqc_cut_merging_cost(w_trial, w_max, s_trial, s_max, K_trial, K_t))


def tqc_choose_slice_cuts(net, mode: int = MODE_STATES, max_log2_input_floats: int = 62,
                          max_log2_intermediate_floats: int = 62, batch_hint: int = 0):
    """The paper's two-level slicing choice (include/tqc.h): list of cut ids in pick order."""
    desc, _keep = _network_desc(net)
    opts = _PlanOpts(mode, 0, None, 0, 0, batch_hint, 0, 0, 0, 0, None, 0, 0)
    out = np.zeros(max(1, len(net.cuts)), dtype=np.int32)
    n = c_int32(0)
    _check(_lib.tqc_choose_slice_cuts(byref(desc), byref(opts), max_log2_input_floats, max_log2_intermediate_floats,
                                      out.ctypes.data, byref(n)))
    return [int(x) for x in out[:n.value]]


def tqc_load_subcircuit_tensors(plan: Plan, s: int, data, stream=None) -> None:
    """data: [4^{c_s}][2^{o_s}] fp32 — a numpy array / CPU torch tensor (HOST) or a CUDA torch tensor (DEVICE)."""
    import torch
    if isinstance(data, torch.Tensor):
        t = data.contiguous()
        if t.dtype != torch.float32:
            raise TypeError("subcircuit tensors must be float32")
        _check(_lib.tqc_load_subcircuit_tensors(plan._h, s, t.data_ptr(), t.numel(), 1 if t.is_cuda else 0,
                                                _stream_ptr(stream)))
        if not t.is_cuda:
            torch.cuda.current_stream().synchronize()      # pageable host source: keep it alive until copied
        return
    a = np.ascontiguousarray(data)
    if a.dtype != np.float32:
        raise TypeError("subcircuit tensors must be float32")
    _check(_lib.tqc_load_subcircuit_tensors(plan._h, s, a.ctypes.data, a.size, 0, _stream_ptr(stream)))
    torch.cuda.current_stream().synchronize()


def tqc_contract_states(plan: Plan, states, out=None, workspace=None, stream=None):
    """states: CUDA int64/uint64 tensor [B, ceil(n/64)] (reading G5).  Returns out (CUDA fp32 [B])."""
    import torch
    if not states.is_cuda or states.element_size() != 8:
        raise TypeError("states must be a CUDA tensor of 64-bit words")
    states = states.contiguous()
    B = states.shape[0]
    if out is None:
        out = torch.empty(B, dtype=torch.float32, device=states.device)
    if workspace is None:
        workspace = torch.empty(plan.workspace_bytes(B), dtype=torch.uint8, device=states.device)
    _check(_lib.tqc_contract_states(plan._h, states.data_ptr(), B, out.data_ptr(), workspace.data_ptr(),
                                    workspace.numel() * workspace.element_size(), _stream_ptr(stream)))
    return out


def tqc_contract_distribution(plan: Plan, prefix_value: int = 0, prefix_bits: int = 0, out=None, workspace=None,
                              stream=None, device="cuda"):
    """Returns out (CUDA fp32 [2^{n - prefix_bits}]), qubit 0 = MSB (reading G4)."""
    import torch
    n = plan.n_qubits
    if out is None:
        out = torch.empty(1 << max(0, n - prefix_bits), dtype=torch.float32, device=device)
    if workspace is None:
        workspace = torch.empty(max(256, plan.workspace_bytes(0, prefix_bits)), dtype=torch.uint8, device=device)
    _check(_lib.tqc_contract_distribution(plan._h, prefix_value, prefix_bits, out.data_ptr(), workspace.data_ptr(),
                                          workspace.numel() * workspace.element_size(), _stream_ptr(stream)))
    return out


def tqc_contract_states_host(plan: Plan, states_host, out_host, workspace, stream=None):
    """End-to-end form: states_host CPU (pinned) 64-bit tensor [B, ceil(n/64)], out_host CPU (pinned) fp32 [B];
    workspace a CUDA uint8 tensor of plan.workspace_bytes_host(B).  Asynchronous on the stream."""
    if states_host.is_cuda or out_host.is_cuda or states_host.element_size() != 8:
        raise TypeError("states_host/out_host must be CPU tensors (64-bit words / float32)")
    B = states_host.shape[0]
    _check(_lib.tqc_contract_states_host(plan._h, states_host.data_ptr(), B, out_host.data_ptr(), workspace.data_ptr(),
                                         workspace.numel() * workspace.element_size(), _stream_ptr(stream)))
    return out_host


def tqc_contract_distribution_host(plan: Plan, out_host, workspace, prefix_value: int = 0, prefix_bits: int = 0,
                                   stream=None):
    """End-to-end form of tqc_contract_distribution: the result lands in out_host (CPU, pinned, fp32)."""
    if out_host.is_cuda:
        raise TypeError("out_host must be a CPU tensor")
    _check(_lib.tqc_contract_distribution_host(plan._h, prefix_value, prefix_bits, out_host.data_ptr(),
                                               workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                                               _stream_ptr(stream)))
    return out_host


def tqc_hss_scores(plan: Plan, s: int, out=None, stream=None, device="cuda"):
    """||p_{s,i}|| for every binary state i of subcircuit s (Alg. 1): CUDA fp32 [2^{o_s}]."""
    import torch
    _, o = plan.tensor_shape(s)
    if out is None:
        out = torch.empty(1 << o, dtype=torch.float32, device=device)
    _check(_lib.tqc_hss_scores(plan._h, s, out.data_ptr(), _stream_ptr(stream)))
    return out


def tqc_hss_select(plan: Plan, scores_host, s_max: int):
    """Alg. 1 lines 480-491 on host score arrays (one float32 numpy array per subcircuit).  Returns x_j as a list of
    int32 arrays, each ascending."""
    import numpy as np
    m = plan.m
    arrs = [np.ascontiguousarray(a, dtype=np.float32) for a in scores_host]
    if len(arrs) != m or any(a.size != 1 << plan.tensor_shape(j)[1] for j, a in enumerate(arrs)):
        raise ValueError("one score array of 2^{o_j} entries per subcircuit")
    ptrs = (c_void_p * m)(*[a.ctypes.data for a in arrs])
    counts = np.zeros(m, dtype=np.int32)
    keys = np.zeros(sum(a.size for a in arrs), dtype=np.int32)
    _check(_lib.tqc_hss_select(plan._h, ptrs, s_max, counts.ctypes.data, keys.ctypes.data, keys.size))
    ofs = np.concatenate([[0], np.cumsum(counts)])
    return [keys[ofs[j]:ofs[j + 1]].copy() for j in range(m)]


def tqc_hss_expand(plan: Plan, x):
    """The prod_j |x_j| composite states of a selection, packed as tqc_contract_states takes them:
    numpy uint64 [B, ceil(n/64)], product order with subcircuit 0 slowest."""
    import numpy as np
    counts = np.array([len(k) for k in x], dtype=np.int32)
    keys = np.ascontiguousarray(np.concatenate([np.asarray(k, dtype=np.int32) for k in x]) if len(x) else
                                np.zeros(0, np.int32))
    n = c_size_t(0)
    _check(_lib.tqc_hss_expand(plan._h, counts.ctypes.data, keys.ctypes.data, None, 0, ctypes.byref(n)))
    words = (plan.n_qubits + 63) // 64
    states = np.zeros((n.value, words), dtype=np.uint64)
    _check(_lib.tqc_hss_expand(plan._h, counts.ctypes.data, keys.ctypes.data, states.ctypes.data, n.value,
                               ctypes.byref(n)))
    return states


def tqc_hss_contract(plan: Plan, x, out=None, workspace=None, stream=None, device="cuda"):
    """Product-structured contraction of a selection x (list of key arrays, as tqc_hss_select returns): CUDA fp32
    [prod_j |x_j|] in the order of tqc_hss_expand, every intermediate shared between the composite states."""
    import torch
    counts = np.array([len(k) for k in x], dtype=np.int32)
    keys = torch.from_numpy(np.ascontiguousarray(np.concatenate([np.asarray(k, dtype=np.int32) for k in x]))).to(device)
    _check(_lib.tqc_hss_prepare(plan._h, counts.ctypes.data, keys.data_ptr(), _stream_ptr(stream)))
    n = int(np.prod(counts.astype(np.int64)))
    if out is None:
        out = torch.empty(n, dtype=torch.float32, device=device)
    if workspace is None:
        workspace = torch.empty(max(256, int(_lib.tqc_hss_workspace_bytes(plan._h))), dtype=torch.uint8, device=device)
    _check(_lib.tqc_hss_contract(plan._h, out.data_ptr(), workspace.data_ptr(), workspace.numel(), _stream_ptr(stream)))
    return out


def tqc_static_scratch_bytes() -> int:
    return int(_lib.tqc_static_scratch_bytes())


def tqc_simulate_subcircuit_tensor_static(w, gates, D_wires, U_wires, O_wires, bond_pos, out, stream=None, fuse_gates=True,
                                          walk_settings=True):
    """tqc_simulate_subcircuit_tensor without a workspace and without any device allocation (tqc.h: "Callers that cannot
    allocate"): `out` is the caller's CUDA fp32 [4^{d+u}, 2^o] tensor, the kernel's scratch is the library's static 8 MiB
    array.  TqcError(TQC_E_TOO_LARGE) when the subcircuit needs more scratch than that."""
    desc, _keep = _subcircuit_desc(w, gates, D_wires, U_wires, O_wires, bond_pos, fuse_gates, walk_settings)
    _check(_lib.tqc_simulate_subcircuit_tensor_static(byref(desc), out.data_ptr(), _stream_ptr(stream)))
    return out


def _subcircuit_desc(w, gates, D_wires, U_wires, O_wires, bond_pos, fuse_gates=True, walk_settings=True):
    garr = _gate_array(gates)
    keep = [garr] + [_i32(v) for v in (D_wires, U_wires, O_wires, bond_pos)]
    desc = _SubcircuitDesc(int(w), len(gates), garr, len(D_wires), len(U_wires), len(O_wires), 1 if fuse_gates else 0,
                           *[ptr for (_arr, ptr) in keep[1:]], 1 if walk_settings else 0, 0)
    return desc, keep


def tqc_simulate_workspace_bytes(w, gates, D_wires, U_wires, O_wires, bond_pos) -> int:
    desc, _keep = _subcircuit_desc(w, gates, D_wires, U_wires, O_wires, bond_pos)
    return int(_lib.tqc_simulate_workspace_bytes(byref(desc)))


def tqc_simulate_subcircuit_tensor(w, gates, D_wires, U_wires, O_wires, bond_pos, out=None, workspace=None, stream=None,
                                   device="cuda", fuse_gates=True, walk_settings=True):
    """T_s of one subcircuit from a device simulation of its 4^d 3^u variants (section 2.1): CUDA fp32
    [4^{d+u}, 2^o] in the layout tqc_load_subcircuit_tensors takes.  gates: (name, params, local wires) in order;
    bond_pos[j]: digit position (0 = most significant) of bond j (D_wires, then U_wires) in the row index."""
    import torch
    desc, _keep = _subcircuit_desc(w, gates, D_wires, U_wires, O_wires, bond_pos, fuse_gates, walk_settings)
    c, o = len(D_wires) + len(U_wires), len(O_wires)
    if out is None:
        out = torch.empty((4 ** c, 2 ** o), dtype=torch.float32, device=device)
    if workspace is None:
        workspace = torch.empty(max(256, int(_lib.tqc_simulate_workspace_bytes(byref(desc)))), dtype=torch.uint8,
                                device=device)
    _check(_lib.tqc_simulate_subcircuit_tensor(byref(desc), out.data_ptr(), workspace.data_ptr(), workspace.numel(),
                                               _stream_ptr(stream)))
    return out
