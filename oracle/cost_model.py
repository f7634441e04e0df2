"""Hybrid cost model of PAPER.md section 5 (lines 509-549) — ORACLE-SIDE (test infrastructure), plain Python.

Eq. 4:  T_QPU = sum_i 3^{u_i} 4^{d_i} 2^{w_i} (t_i t_g + t_m), with t_g = 1e-7 s per gate layer and
t_m = 1e-6 s per measurement; the 2^{w_i} factor is the number of shots, "equal to the number of quantum
states per subcircuit, with limits ranging from 2^10 to 2^20"; more QPUs divide it linearly (the
experiments assume 10).  Eq. 5: T_classical = C_TN / FLOPs.  Eq. 6: T = T_QPU + T_classical.
Pinned by a hand-worked example (tests/golden/cost_model.txt).
"""
from __future__ import annotations


def t_qpu(subcircuits, t_g: float = 1e-7, t_m: float = 1e-6, n_qpus: int = 10, shots_log2=(10, 20)) -> float:
    """subcircuits: iterable of (u_i, d_i, w_i, t_i)."""
    lo, hi = shots_log2
    total = 0.0
    for (u, d, w, t) in subcircuits:
        shots = 2.0 ** min(max(w, lo), hi)
        total += (3.0 ** u) * (4.0 ** d) * shots * (t * t_g + t_m)
    return total / n_qpus


def t_classical(c_tn_flop: float, flops: float) -> float:
    return c_tn_flop / flops


def t_total(subcircuits, c_tn_flop: float, flops: float, **kw) -> float:
    return t_qpu(subcircuits, **kw) + t_classical(c_tn_flop, flops)
