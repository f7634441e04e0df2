"""The allocation-free entry point (include/tqc.h: "Callers that cannot allocate"): tqc_simulate_subcircuit_tensor_static
against the existing tqc_simulate_subcircuit_tensor, on two calls in a row.

Named test_zz_* so that pytest collects it LAST (the suite runs with `pytest -x`).  Both entry points run the same kernels
in fp64 and round once to fp32, so they should agree exactly; the assertion uses the tolerance of tests/test_gpu_variants.py
(2^{d_s} * 2^-24, doubled: 2^{d_s - 23}).  The static array is shared between calls and keeps the last call's contents, so
the second call uses a DIFFERENT, smaller subcircuit (a stale value of the first call would show), then the first subcircuit
is run once more.
"""
import numpy as np
import pytest
import torch

import paper_2502_03445_b200 as tqc
from tqc_inputs.circuits import hea_subcircuit

pytestmark = pytest.mark.gpu


def _both(desc, d):
    c, o = len(desc["D_wires"]) + len(desc["U_wires"]), len(desc["O_wires"])
    want = tqc.tqc_simulate_subcircuit_tensor(**desc)                        # existing path: caller's workspace
    out = torch.full((4 ** c, 2 ** o), float("nan"), dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    got = tqc.tqc_simulate_subcircuit_tensor_static(**desc, out=out)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    err = (got.double() - want.double()).abs().max().item()
    assert err <= 2.0 ** (d - 23), err
    assert bool(torch.isfinite(got).all())
    return free0, free1


def test_static_scratch_entry_point_matches_the_workspace_path_on_two_calls_in_a_row():
    assert tqc.tqc_static_scratch_bytes() == 8 << 20
    big = hea_subcircuit(10, 2, 2, seed=77)                   # R = 4^4 * 2^8 doubles = 512 KB
    small = hea_subcircuit(6, 1, 2, seed=78)                  # R = 4^3 * 2^4 doubles = 8 KB: the front of the same array
    assert 0 < tqc.tqc_simulate_workspace_bytes(**big) <= tqc.tqc_static_scratch_bytes()
    _both(big, 2)                                             # first call: may load kernels (lazy module loading)
    f0, f1 = _both(small, 1)                                  # second call, right after the first, on the same array
    assert f1 >= f0, ("the call took device memory", f0, f1)
    f0, f1 = _both(big, 2)
    assert f1 >= f0, ("the call took device memory", f0, f1)


def test_static_scratch_rejects_what_does_not_fit():
    desc = hea_subcircuit(14, 2, 2, seed=1414)                # amplitudes in the workspace: far beyond 8 MiB
    assert tqc.tqc_simulate_workspace_bytes(**desc) > tqc.tqc_static_scratch_bytes()
    out = torch.zeros((4 ** 4, 2 ** 12), dtype=torch.float32, device="cuda")
    with pytest.raises(tqc.TqcError) as e:
        tqc.tqc_simulate_subcircuit_tensor_static(**desc, out=out)
    assert e.value.code == -6 and "static array holds" in str(e.value)
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0                      # nothing was launched
    with pytest.raises(tqc.TqcError) as e:                    # R alone = 4^6 * 2^9 doubles = 16 MiB
        tqc.tqc_simulate_subcircuit_tensor_static(**hea_subcircuit(12, 3, 3), out=torch.zeros((4 ** 6, 2 ** 9), device="cuda"))
    assert e.value.code == -6
