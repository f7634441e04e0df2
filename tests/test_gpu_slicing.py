"""GPU parity of index slicing (Fig. 6) through the C ABI: a plan with slice_cuts evaluates the
4^{|S|} smaller networks and sums them.  Checked against the oracle's sliced_sum / direct sum (|dp| <= 1e-5 max p), against
the unsliced GPU plan, in both modes, with a chunked workspace, and on a network whose first step runs on the tensor pipe."""
import numpy as np
import pytest
import torch

import paper_2502_03445_b200 as tqc
from oracle import reconstruct as R
from oracle.direct_sum_c import direct_sum_c
from tqc_inputs import configs, pack_states, random_states, random_tensors
from tqc_inputs.network import Network

pytestmark = pytest.mark.gpu
TOL = 1e-5


def _loaded(net, T, mode, **kw):
    plan = tqc.tqc_plan(net, mode, **kw)
    for s, t in enumerate(T):
        tqc.tqc_load_subcircuit_tensors(plan, s, np.ascontiguousarray(t, dtype=np.float32))
    return plan


def _states(plan, bits, workspace=None):
    out = tqc.tqc_contract_states(plan, torch.from_numpy(pack_states(bits).view(np.int64)).cuda(), workspace=workspace)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("seed,slice_cuts", [(0, [1]), (1, [0, 4]), (2, [5, 2, 3]), (3, [6, 0])])
def test_sliced_states_match_oracle(seed, slice_cuts):
    net = configs.random_network(3 + seed, 7, seed=300 + seed, o_lo=0, o_hi=4)
    T = [np.asarray(t, dtype=np.float32) for t in random_tensors(net, 310 + seed)]
    if seed == 2:
        rng = np.random.default_rng(5)
        T = [(rng.random(t.shape) * 2 - 1).astype(np.float32) for t in T]            # signed values
    bits = random_states(net.n_qubits, 777, 320 + seed)
    plan = _loaded(net, T, tqc.MODE_STATES, slice_cuts=slice_cuts, batch_hint=777)
    got = _states(plan, bits)
    want = R.direct_sum(net, T, bits)
    assert np.abs(got - want).max() <= TOL * np.abs(want).max()
    assert np.allclose(R.sliced_sum(net, T, bits[:16], slice_cuts), want[:16], rtol=1e-12)
    whole = _states(_loaded(net, T, tqc.MODE_STATES, batch_hint=777), bits)
    assert np.abs(got - whole).max() <= TOL * np.abs(want).max()
    # a workspace that forces several chunks (partial-sum buffer + minimum + a little)
    small = torch.empty(plan.workspace_min_bytes() + 4 * 777 + 256 + 150 * 64, dtype=torch.uint8, device="cuda")
    assert np.array_equal(_states(plan, bits, workspace=small), got)
    # the advertised minimum is enough (include/tqc.h): the batch is then cut into pieces, each summed over all sub-networks
    tiny = torch.empty(plan.workspace_min_bytes(), dtype=torch.uint8, device="cuda")
    assert np.array_equal(_states(plan, bits, workspace=tiny), got)
    # reloading a tensor replaces every slice of it
    T2 = [t.copy() for t in T]
    T2[0] = T2[0][::-1].copy()
    tqc.tqc_load_subcircuit_tensors(plan, 0, T2[0])
    want2 = R.direct_sum(net, T2, bits[:64])
    assert np.abs(_states(plan, bits)[:64] - want2).max() <= TOL * np.abs(want2).max()


def test_sliced_distribution_and_prefix():
    net = configs.random_network(4, 6, seed=401, o_lo=1, o_hi=4)
    T = [np.asarray(t, dtype=np.float32) for t in random_tensors(net, 402)]
    want = R.direct_sum(net, T, R.full_distribution_bits(net.n_qubits))
    plan = _loaded(net, T, tqc.MODE_DISTRIBUTION, slice_cuts=[2, 5])
    out = tqc.tqc_contract_distribution(plan)
    torch.cuda.synchronize()
    assert np.abs(out.cpu().numpy() - want).max() <= TOL * want.max()
    pb = 3
    for pv in (0, 5):
        part = tqc.tqc_contract_distribution(plan, pv, pb)
        torch.cuda.synchronize()
        n_out = 1 << (net.n_qubits - pb)
        assert np.abs(part.cpu().numpy() - want[pv * n_out:(pv + 1) * n_out]).max() <= TOL * want.max()


def test_sliced_plan_with_tensor_pipe_step_and_host_buffers():
    """Triangle A-B-D with 5 + 2 + 3 cuts: slicing one A-D cut leaves M = 4^4, N = 4^2, K = 4^3 per state (tcgen05 step)."""
    cuts = [(0, 2)] * 5 + [(2, 1)] * 2 + [(0, 1)] * 3
    net = Network(8, cuts, [[0, 1, 2, 3, 4, 7, 8, 9], [5, 6, 7, 8, 9], [0, 1, 2, 3, 4, 5, 6]], [[0, 1, 2], [3, 4, 5], [6, 7]])
    net.validate()
    T = [np.asarray(t, dtype=np.float32) for t in random_tensors(net, 17)]
    bits = random_states(8, 200, 19)
    plan = _loaded(net, T, tqc.MODE_STATES, slice_cuts=[1], order=[(0, 1), (3, 2)], batch_hint=4)
    assert plan.step(0)["kernel_class"] == 2
    want, _ = direct_sum_c(net, T, bits)
    got = _states(plan, bits)
    assert np.abs(got - want).max() <= TOL * want.max()
    sh = torch.from_numpy(pack_states(bits).view(np.int64)).pin_memory()
    oh = torch.empty(200, dtype=torch.float32).pin_memory()
    ws = torch.empty(plan.workspace_bytes_host(200), dtype=torch.uint8, device="cuda")
    tqc.tqc_contract_states_host(plan, sh, oh, ws)
    torch.cuda.synchronize()
    assert np.array_equal(oh.numpy().astype(np.float64), got)
    with pytest.raises(tqc.TqcError):
        tqc.tqc_hss_scores(plan, 0)


def test_two_level_choice_end_to_end():
    """tqc_choose_slice_cuts -> tqc_plan(slice_cuts) -> contract: limits met and the values are still Eq. 1."""
    net = configs.random_network(6, 11, seed=611, o_lo=1, o_hi=3)
    T = [np.asarray(t, dtype=np.float32) for t in random_tensors(net, 612)]
    bits = random_states(net.n_qubits, 500, 613)
    full = tqc.tqc_plan(net, tqc.MODE_STATES, use_chain=-1)
    inter = max(2 * full.node(net.m + t)["n_open"] for t in range(net.m - 1))
    big_in = max(2 * net.c(s) + net.o(s) for s in range(net.m))
    cuts = tqc.tqc_choose_slice_cuts(net, tqc.MODE_STATES, big_in - 2, max(inter - 4, 2))
    assert len(cuts) >= 2
    plan = _loaded(net, T, tqc.MODE_STATES, slice_cuts=cuts)
    assert max(2 * plan.node(net.m + t)["n_open"] for t in range(net.m - 1)) <= max(inter - 4, 2)
    want, _ = direct_sum_c(net, T, bits)
    got = _states(plan, bits)
    assert np.abs(got - want).max() <= TOL * want.max()
