"""GPU parity: libtqc.so (through the C ABI) against the CPU oracle, element by element.

Bar (BASELINE.json north_star): |dp| <= 1e-5 * max_x p(x), max over the oracle-evaluated set
(reading G8); bit-exact state indexing (each out[b] belongs to the caller's b).
"""
import numpy as np
import pytest
import torch

import paper_2502_03445_b200 as tqc
from oracle import cutting, reconstruct as R, statevector as sv
from oracle.direct_sum_c import direct_sum_c
from tqc_inputs import configs, pack_states, random_states, random_tensors, rank_one_tensors, seed_for
from tqc_inputs.network import Network
from tqc_inputs.seeds import STREAM_STATES, STREAM_SUBSET, STREAM_TENSORS

pytestmark = pytest.mark.gpu
TOL = 1e-5          # north_star: |dp| <= 1e-5 * max p


def _loaded_plan(net, tensors, mode, **kw):
    plan = tqc.tqc_plan(net, mode, **kw)
    for s, t in enumerate(tensors):
        tqc.tqc_load_subcircuit_tensors(plan, s, np.ascontiguousarray(t, dtype=np.float32))
    return plan


def _states_dev(bits):
    return torch.from_numpy(pack_states(bits).view(np.int64)).cuda()


def _gpu_states(net, tensors, bits, workspace_bytes=None, **kw):
    plan = _loaded_plan(net, tensors, tqc.MODE_STATES, **kw)
    st = _states_dev(bits)
    ws = None
    if workspace_bytes is not None:
        ws = torch.empty(workspace_bytes, dtype=torch.uint8, device="cuda")
    out = tqc.tqc_contract_states(plan, st, workspace=ws)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64), plan


def _gpu_distribution(net, tensors, prefix_value=0, prefix_bits=0, **kw):
    plan = _loaded_plan(net, tensors, tqc.MODE_DISTRIBUTION, **kw)
    out = tqc.tqc_contract_distribution(plan, prefix_value, prefix_bits)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64), plan


def _assert_close(got, want):
    assert got.shape == want.shape
    err = np.abs(got - want).max() if got.size else 0.0
    assert err <= TOL * np.abs(want).max(), (err, np.abs(want).max())


def _f32(tensors):
    """The library consumes fp32; the oracle gets the same values widened exactly."""
    return [np.asarray(t, dtype=np.float32) for t in tensors]


# ---- small random networks: every kernel path, ragged batches, axis-order shuffles ------------
@pytest.mark.parametrize("seed", range(24))
def test_states_random_networks(seed):
    m = 1 + seed % 6
    K = 0 if m == 1 else m - 1 + seed % 4
    net = configs.random_network(m, K, 500 + seed, o_lo=0, o_hi=3, connected=(seed % 5 != 0))
    T = random_tensors(net, 600 + seed)
    B = [1, 37, 64, 257, 1000, 4099][seed % 6]
    bits = random_states(net.n_qubits, B, 700 + seed)
    want = R.direct_sum(net, T, bits)
    for hint in (0, 4):                       # default (tables where possible) and per-state evaluation
        for chain in (0, -2, -1):             # fused chain kernel specialised for the plan / generic / one kernel per step
            got, _ = _gpu_states(net, T, bits, batch_hint=hint, use_chain=chain)
            _assert_close(got, want)


@pytest.mark.parametrize("seed", range(16))
def test_distribution_random_networks(seed):
    m = 1 + seed % 5
    K = 0 if m == 1 else m - 1 + seed % 3
    net = configs.random_network(m, K, 800 + seed, o_lo=0, o_hi=3, connected=(seed % 5 != 0))
    T = random_tensors(net, 900 + seed)
    n = net.n_qubits
    want = R.direct_sum(net, T, R.full_distribution_bits(n))
    got, _ = _gpu_distribution(net, T)
    _assert_close(got, want)
    if n >= 2:                                # output-bit slicing: a fixed prefix gives the matching chunk
        g = 1 + seed % min(n, 3)
        for pv in range(1 << g):
            chunk, _ = _gpu_distribution(net, T, prefix_value=pv, prefix_bits=g)
            lo = pv << (n - g)
            assert np.abs(chunk - want[lo:lo + (1 << (n - g))]).max() <= TOL * np.abs(want).max()


def test_signed_tensors_and_cancellation():
    """Real-circuit tensors are signed (|T| <= 2^{d_s}, reading G16): use signed values."""
    net = configs.random_network(5, 7, 4242, o_lo=1, o_hi=3)
    rng = np.random.default_rng(5)
    T = [(rng.random(net.tensor_shape(s)) * 2 - 1).astype(np.float32) for s in range(net.m)]
    bits = random_states(net.n_qubits, 3001, 6)
    want = R.direct_sum(net, T, bits)
    got, _ = _gpu_states(net, T, bits)
    _assert_close(got, want)


def test_state_indexing_duplicates_and_chunking():
    """Duplicates are legal, every index gets its own output (G5); a small workspace chunks the
    batch without changing any value (bit-exact across chunk sizes)."""
    net = configs.random_network(5, 8, 77, o_lo=2, o_hi=3)
    T = random_tensors(net, 78)
    bits = random_states(net.n_qubits, 5000, 79)
    bits[100:200] = bits[0:100]
    full, plan = _gpu_states(net, T, bits, batch_hint=4)
    assert np.array_equal(full[100:200], full[0:100])
    small = plan.workspace_min_bytes() + 4096
    chunked, _ = _gpu_states(net, T, bits, workspace_bytes=small, batch_hint=4)
    assert np.array_equal(full, chunked)
    _assert_close(full, R.direct_sum(net, T, bits))


def test_empty_batch_and_errors():
    net = configs.random_network(3, 3, 11, o_lo=1, o_hi=2)
    T = random_tensors(net, 12)
    plan = tqc.tqc_plan(net)
    st = _states_dev(random_states(net.n_qubits, 8, 1))
    with pytest.raises(tqc.TqcError) as e:                      # tensors not loaded
        tqc.tqc_contract_states(plan, st)
    assert e.value.code == -3
    with pytest.raises(tqc.TqcError) as e:                      # wrong shape
        tqc.tqc_load_subcircuit_tensors(plan, 0, np.zeros(3, dtype=np.float32))
    assert e.value.code == -2
    for s, t in enumerate(T):
        tqc.tqc_load_subcircuit_tensors(plan, s, t)
    out = tqc.tqc_contract_states(plan, st[:0])
    assert out.numel() == 0
    with pytest.raises(tqc.TqcError) as e:                      # states plan used for a distribution
        tqc.tqc_contract_distribution(plan)
    assert e.value.code == -3


def test_device_resident_tensor_load_equals_host_load():
    net = configs.random_network(4, 5, 21, o_lo=2, o_hi=3)
    T = random_tensors(net, 22)
    bits = random_states(net.n_qubits, 513, 23)
    a, _ = _gpu_states(net, T, bits)
    plan = tqc.tqc_plan(net)
    for s, t in enumerate(T):
        tqc.tqc_load_subcircuit_tensors(plan, s, torch.from_numpy(t).cuda())
    b = tqc.tqc_contract_states(plan, _states_dev(bits)).cpu().numpy().astype(np.float64)
    assert np.array_equal(a, b)


def test_order_invariance_on_gpu():
    """Any contraction order gives the same value, to fp32 rounding."""
    net = Network(4, [(0, 1), (1, 2), (1, 3), (2, 3)], [[0], [0, 1, 2], [1, 3], [2, 3]], [[0], [1], [2], [3]])
    T = random_tensors(net, 31)
    bits = R.full_distribution_bits(4)
    want = R.direct_sum(net, T, bits)
    for order in ([(0, 1), (4, 2), (5, 3)], [(2, 3), (4, 1), (5, 0)], [(1, 2), (0, 3), (4, 5)]):
        got, _ = _gpu_states(net, T, bits, order=order)
        _assert_close(got, want)


def test_host_buffer_entry_points_and_profile_hooks():
    """tqc_contract_states_host / tqc_contract_distribution_host (pinned HOST buffers, the end-to-end form bench.py times)
    give the same values as the device-pointer calls; the per-launch profile returns one entry per kernel launch."""
    net = configs.random_network(5, 7, 91, o_lo=1, o_hi=3)
    T = random_tensors(net, 92)
    bits = random_states(net.n_qubits, 777, 93)
    dev, plan = _gpu_states(net, T, bits)
    sh = torch.from_numpy(pack_states(bits).view(np.int64)).pin_memory()
    oh = torch.empty(bits.shape[0], dtype=torch.float32).pin_memory()
    ws = torch.empty(plan.workspace_bytes_host(bits.shape[0]), dtype=torch.uint8, device="cuda")
    plan.profile_enable(True)
    l0 = plan.launch_count
    tqc.tqc_contract_states_host(plan, sh, oh, ws)
    torch.cuda.synchronize()
    prof = plan.profile_read()
    plan.profile_enable(False)
    assert np.array_equal(oh.numpy().astype(np.float64), dev)
    assert len(prof) == plan.launch_count - l0 and all(ms >= 0 for _, ms in prof)
    ddev, pland = _gpu_distribution(net, T)
    dh = torch.empty(1 << net.n_qubits, dtype=torch.float32).pin_memory()
    wsd = torch.empty(pland.workspace_bytes_host(0, 0), dtype=torch.uint8, device="cuda")
    tqc.tqc_contract_distribution_host(pland, dh, wsd)
    torch.cuda.synchronize()
    assert np.array_equal(dh.numpy().astype(np.float64), ddev)


@pytest.mark.parametrize("net_name", ["cfg4", "rand"])
def test_host_buffer_pipeline_large_batch(net_name):
    """A large ragged batch through tqc_contract_states_host on a non-default stream: the table steps are forked off
    before the host-to-device copy.  Same values as the device-pointer call, repeated calls on the same buffers (the
    staging area is reused), and the caller's stream order covering the copy back."""
    if net_name == "cfg4":
        net = configs.cfg4_network()
    else:
        net = configs.random_network(5, 7, 191, o_lo=2, o_hi=4)
    T = random_tensors(net, 192)
    plan = _loaded_plan(net, T, tqc.MODE_STATES, batch_hint=1 << 17)
    B = 70001
    ws = torch.empty(plan.workspace_bytes_host(B), dtype=torch.uint8, device="cuda")
    oh = torch.empty(B, dtype=torch.float32).pin_memory()
    stream = torch.cuda.Stream()
    for rep in range(3):
        bits = random_states(net.n_qubits, B, 193 + rep)
        sh = torch.from_numpy(pack_states(bits).view(np.int64)).pin_memory()
        oh.fill_(-1.0)
        with torch.cuda.stream(stream):
            tqc.tqc_contract_states_host(plan, sh, oh, ws, stream=stream)
        stream.synchronize()                                  # only the caller's stream: the side streams must be joined
        got = oh.numpy().copy()
        dev = tqc.tqc_contract_states(plan, sh.cuda())
        torch.cuda.synchronize()
        assert np.array_equal(got, dev.cpu().numpy())
    want = direct_sum_c(net, T, bits[:24])[0] if net_name == "cfg4" else R.direct_sum(net, T, bits[:200])
    assert np.abs(got[:len(want)] - want).max() <= TOL * np.abs(want).max()
