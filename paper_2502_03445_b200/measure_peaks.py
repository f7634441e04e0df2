"""Measures the roofline denominators that MEASURED_PEAKS.json lacks on the current GPU and writes them
as JSON:  python -m paper_2502_03445_b200.measure_peaks [out.json]

  tf32_tflops / tf32_tflops_sustained   torch.matmul fp32 8192^3 with TF32 enabled (cuBLAS): best of 10, and back to back for 3 s
  ffma_tflops                           register-resident FFMA loop on every SM (csrc/peaks.cu), >= 1 s
  lds_gbs                               conflict-free LDS.128 loop on every SM
  l2_read_gbs                           32 MB buffer read repeatedly (ld.global.cg)
  store_gbs                             the store path by warp pattern and row pitch (the pair kernel's epilogue)
bench.py reads the committed copy (profiles/peaks_r02.json) for the `peak` of its alu / tensor / smem rooflines.
"""
from __future__ import annotations

import ctypes
import json
import os
import sys
import time

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(_HERE, "libtqc_peaks.so")


def measure() -> dict:
    import torch
    lib = ctypes.CDLL(LIB)
    dbl = ctypes.c_double
    out = {"gpu": torch.cuda.get_device_name(0), "when": time.strftime("%Y-%m-%dT%H:%M:%SZ", time.gmtime())}
    # TF32 dense matmul through cuBLAS
    torch.backends.cuda.matmul.allow_tf32 = True
    n = 8192
    a = torch.randn(n, n, device="cuda")
    b = torch.randn(n, n, device="cuda")
    for _ in range(3):
        a @ b
    torch.cuda.synchronize()
    best = 1e9
    for _ in range(10):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); a @ b; e1.record(); torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    out["tf32_tflops"] = 2.0 * n ** 3 / (best * 1e-3) / 1e12
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = max(10, int(3000.0 / best))
    e0.record()
    for _ in range(reps):
        a @ b
    e1.record(); torch.cuda.synchronize()
    out["tf32_tflops_sustained"] = 2.0 * n ** 3 * reps / (e0.elapsed_time(e1) * 1e-3) / 1e12
    torch.backends.cuda.matmul.allow_tf32 = False
    del a, b
    v, ms = dbl(), dbl()
    assert lib.tqc_peak_ffma(1 << 17, ctypes.byref(v), ctypes.byref(ms)) == 0
    out["ffma_tflops"], out["ffma_ms"] = v.value, ms.value
    assert lib.tqc_peak_lds(1 << 17, ctypes.byref(v), ctypes.byref(ms)) == 0
    out["lds_gbs"], out["lds_ms"] = v.value, ms.value
    lib.tqc_peak_l2.argtypes = [ctypes.c_size_t, ctypes.c_int, ctypes.POINTER(dbl), ctypes.POINTER(dbl)]
    assert lib.tqc_peak_l2(32 << 20, 2000, ctypes.byref(v), ctypes.byref(ms)) == 0
    out["l2_read_gbs"], out["l2_ms"] = v.value, ms.value
    # store path by warp pattern and row pitch: 16 GB written once, one 512-thread block per SM, and one SM alone
    lib.tqc_peak_store.argtypes = [ctypes.c_int, ctypes.c_size_t, ctypes.c_size_t, ctypes.c_int, ctypes.POINTER(dbl), ctypes.POINTER(dbl)]
    names = {1: "st.v2 quad = 32 B sector, 8 rows per instruction", 2: "st.v4 8 lanes = 128 B line, 4 rows",
             4: "st.v4 warp = 512 B of one row", 5: "st.v4 quad = 64 B of a row, 8 rows"}
    store = {}
    for pat in (1, 2, 4, 5):
        for pitch in (1024, 16384, 65536, 1 << 20):
            assert lib.tqc_peak_store(pat, 16 << 30, pitch, 0, ctypes.byref(v), ctypes.byref(ms)) == 0
            store[f"pattern {pat} ({names[pat]}), pitch {pitch}"] = round(v.value, 1)
        assert lib.tqc_peak_store(pat, 1 << 30, 16384, 1, ctypes.byref(v), ctypes.byref(ms)) == 0
        store[f"pattern {pat}, ONE block on one SM, pitch 16384"] = round(v.value, 1)
    out["store_gbs"] = store
    out["how"] = ("tf32: torch.matmul fp32 8192^3, allow_tf32, best of 10 / back to back for 3 s; ffma: 8 FMA chains per "
                  "thread, 1024 threads per SM, all SMs; lds: conflict-free LDS.128, 1024 threads per SM; l2: 32 MB buffer, "
                  "ld.global.cg float4, 2048 threads per SM, 2000 passes (csrc/peaks.cu)")
    return out


if __name__ == "__main__":
    res = measure()
    text = json.dumps(res, indent=1)
    print(text)
    if len(sys.argv) > 1:
        with open(sys.argv[1], "w") as f:
            f.write(text + "\n")
