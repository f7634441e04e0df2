"""ctypes wrapper around oracle/direct_sum.c (O6 in C) — ORACLE CODE, test infrastructure."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

from .reconstruct import keys_from_bits

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle_direct_sum.so")
_lib = None


def build(force: bool = False) -> str:
    src = os.path.join(_HERE, "direct_sum.c")
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _SO, src, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.tqc_oracle_direct_sum.restype = ctypes.c_int
    return _lib


def direct_sum_c(net, tensors, bits: np.ndarray, num_threads: int = 0):
    """Returns (p float64 [B], threads used)."""
    lib = _load()
    m, K = net.m, net.K
    keys = np.ascontiguousarray(keys_from_bits(net, bits), dtype=np.int64)
    B = keys.shape[0]
    T = [np.ascontiguousarray(t, dtype=np.float64) for t in tensors]
    ptrs = (ctypes.c_void_p * max(m, 1))(*[t.ctypes.data for t in T])
    ofs = np.zeros(m + 1, dtype=np.int32)
    flat = []
    for s in range(m):
        flat += list(net.sub_cuts[s])
        ofs[s + 1] = len(flat)
    flat = np.asarray(flat if flat else [0], dtype=np.int32)
    two_o = np.asarray([2 ** net.o(s) for s in range(m)], dtype=np.int64)
    out = np.zeros(B, dtype=np.float64)
    used = lib.tqc_oracle_direct_sum(
        ctypes.c_int(m), ctypes.c_int(K), ofs.ctypes.data_as(ctypes.c_void_p),
        flat.ctypes.data_as(ctypes.c_void_p), ptrs, two_o.ctypes.data_as(ctypes.c_void_p),
        keys.ctypes.data_as(ctypes.c_void_p), ctypes.c_int64(B),
        out.ctypes.data_as(ctypes.c_void_p), ctypes.c_int(num_threads))
    return out, int(used)
