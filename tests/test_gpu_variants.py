"""GPU parity of the device variant simulation (tqc_simulate_subcircuit_tensor) against the
oracle's O4/O5 (oracle/cutting.build_tensor, float64) and, end to end, against the UNCUT statevector (O7).

The library gets only the plain subcircuit description (wires, gate names and angles, cut / output wire lists): the
gate matrices, preparation states, measurement rotations and kappa / sigma tables on its side are its own.
Tolerance: the device computes in fp64 and rounds once to fp32; |T_s| <= 2^{d_s} (reading G16), so an entry may differ
from the float64 value by half an fp32 ulp of 2^{d_s}: 2^{d_s} * 2^-24, doubled for slack.
"""
import numpy as np
import pytest
import torch

import paper_2502_03445_b200 as tqc
from oracle import cutting, statevector as sv
from types import SimpleNamespace

from tqc_inputs import circuits as C, configs
from tqc_inputs.circuits import hea_subcircuit

pytestmark = pytest.mark.gpu


def _args(net, sub):
    have = [e for (_w, e) in sub.D] + [e for (_w, e) in sub.U]
    want = list(net.sub_cuts[sub.sid])
    return dict(w=sub.w, gates=sub.gates, D_wires=[w for (w, _e) in sub.D], U_wires=[w for (w, _e) in sub.U],
                O_wires=[w for (w, _q) in sub.O], bond_pos=[want.index(e) for e in have])


def _gpu_tensors(net, subs, fuse=True):
    # fuse = False also turns the settings walk off: one pass per listed gate, one block per variant
    out = [tqc.tqc_simulate_subcircuit_tensor(**_args(net, sub), fuse_gates=fuse, walk_settings=fuse) for sub in subs]
    torch.cuda.synchronize()
    return out


def _check_against_oracle(net, subs, T64, fuse=True):
    got = _gpu_tensors(net, subs, fuse)
    for sub, g, t in zip(subs, got, T64):
        assert tuple(g.shape) == t.shape
        tol = 2.0 ** (len(sub.D) - 23)
        err = np.abs(g.cpu().numpy().astype(np.float64) - t).max()
        assert err <= tol, (sub.sid, err, tol)
    return got


def test_plus_state_fixture():
    # |+> measured at one upstream cut, no outputs -> (I, X, Y, Z) = (1, 1, 0, 0)
    t = tqc.tqc_simulate_subcircuit_tensor(1, [("h", (), (0,))], [], [0], [], [0])
    assert np.abs(t.cpu().numpy().reshape(-1) - np.array([1, 1, 0, 0])).max() < 1e-7
    # |i> = S H |0>: (1, 0, 1, 0); a downstream wire straight to an output: Z basis gives +-1, I gives 1, X and Y give 0
    t = tqc.tqc_simulate_subcircuit_tensor(1, [("h", (), (0,)), ("s", (), (0,))], [], [0], [], [0])
    assert np.abs(t.cpu().numpy().reshape(-1) - np.array([1, 0, 1, 0])).max() < 1e-7
    t = tqc.tqc_simulate_subcircuit_tensor(1, [], [0], [], [0], [0]).cpu().numpy()
    assert np.abs(t - np.array([[1, 1], [0, 0], [0, 0], [1, -1]])).max() < 1e-7
    # a subcircuit no gate was assigned to (w = 0): the empty product, a 1 x 1 tensor [1]   (reading G15)
    assert tqc.tqc_simulate_subcircuit_tensor(0, [], [], [], [], []).cpu().numpy().tolist() == [[1.0]]


def _cut_circuit(n, n2q, m, seed, kmax=6):
    """Seeded rejection loop (same recipe as tests/test_oracle_circuits.py): every part used, 1 <= K <= kmax."""
    for bump in range(400):
        circ = C.random_small_circuit(n, n2q, seed + 7919 * bump)
        C.assign_parts_random(circ, m, seed + 13 * bump)
        if sorted(set(p for p in circ.parts if p is not None)) != list(range(m)):
            continue
        net, subs = cutting.extract(circ)
        if 1 <= net.K <= kmax and max(s.w for s in subs) <= 10:
            return circ
    raise AssertionError("no circuit found")


@pytest.mark.parametrize("seed", range(8))
def test_random_circuits_every_gate_kind(seed):
    circ = _cut_circuit(6 + seed % 4, 8 + seed, 2 + seed % 2, 1000 + seed)
    net, T64, subs = cutting.tensors_from_circuit(circ)
    _check_against_oracle(net, subs, T64, fuse=False)           # one pass per listed gate
    got = _check_against_oracle(net, subs, T64)                 # one-qubit gates folded into their two-qubit neighbours
    # the second construction (O5', no measurement rotations, no kappa table) agrees as well
    _net2, T64b, _ = cutting.tensors_from_circuit(circ, operator_form=True)
    for sub, g, t in zip(subs, got, T64b):
        assert np.abs(g.cpu().numpy().astype(np.float64) - t).max() <= 2.0 ** (len(sub.D) - 23)


@pytest.mark.parametrize("cfg,n", [("cfg1", 8), ("cfg2", 20)])
def test_simulated_tensors_reconstruct_the_uncut_distribution(cfg, n):
    circ = getattr(configs, cfg + "_circuit")()
    net, T64, subs = cutting.tensors_from_circuit(circ)
    got = _check_against_oracle(net, subs, T64)
    plan = tqc.tqc_plan(net, tqc.MODE_DISTRIBUTION)
    for s, t in enumerate(got):
        tqc.tqc_load_subcircuit_tensors(plan, s, t)             # device pointer: nothing touches the host
    p = tqc.tqc_contract_distribution(plan).cpu().numpy().astype(np.float64)
    want = sv.uncut_probabilities(n, circ.gates)
    assert np.abs(p - want).max() <= 1e-5 * want.max()
    assert abs(p.sum() - 1.0) < 1e-4


def test_ghz_closed_form_through_device_tensors():
    # GHZ-10 (P:742-744 benchmark family; closed form S:61): H, CX ladder, three parts -> p(0...0) = p(1...1) = 1/2
    n = 10
    gates = [("h", (), (0,))] + [("cx", (), (q, q + 1)) for q in range(n - 1)]
    circ = C.Circuit(n, gates, name="ghz10")
    C.assign_parts_by_qubit_ranges(circ, [3, 7])
    net, subs = cutting.extract(circ)
    assert net.K >= 2
    plan = tqc.tqc_plan(net, tqc.MODE_DISTRIBUTION)
    for sub, t in zip(subs, _gpu_tensors(net, subs)):
        tqc.tqc_load_subcircuit_tensors(plan, sub.sid, t)
    p = tqc.tqc_contract_distribution(plan).cpu().numpy().astype(np.float64)
    want = np.zeros(1 << n)
    want[0] = want[-1] = 0.5
    assert np.abs(p - want).max() <= 1e-6


def test_cfg3_subcircuits_twelve_wires():
    circ = configs.cfg3_circuit()
    net, T64, subs = cutting.tensors_from_circuit(circ)
    assert max(sub.w for sub in subs) == 12
    _check_against_oracle(net, subs, T64, fuse=False)
    _check_against_oracle(net, subs, T64)


def test_bench_subcircuit_in_the_launch_configuration_bench_times():
    # bench.py's `variants` row: 12 wires, d = u = 3, 576 blocks walking 3 settings each, whole tensor against O4/O5
    from types import SimpleNamespace
    desc = C.hea_subcircuit(12, 3, 3)
    sub = cutting.Subcircuit(0, w=12, gates=desc["gates"], D=[(q, i) for i, q in enumerate(desc["D_wires"])],
                             U=[(q, 3 + j) for j, q in enumerate(desc["U_wires"])], O=[(q, q) for q in desc["O_wires"]])
    want = cutting.build_tensor(SimpleNamespace(sub_cuts=[list(range(6))]), sub)
    for walk in (True, False):
        got = tqc.tqc_simulate_subcircuit_tensor(**desc, walk_settings=walk).cpu().numpy().astype(np.float64)
        assert np.abs(got - want).max() <= 2.0 ** (3 - 23)
    assert abs(want[0].sum() - 8.0) < 1e-9                      # sum_x T[I...I, x] = 2^{d_s}   (reading G16)
    # a permuted axis order is the same tensor with its base-4 digits permuted
    perm = [2, 0, 1, 5, 3, 4]
    got_p = tqc.tqc_simulate_subcircuit_tensor(**{**desc, "bond_pos": perm}).cpu().numpy().astype(np.float64)
    want_p = np.transpose(want.reshape((4,) * 6 + (512,)), list(np.argsort(perm)) + [6]).reshape(4096, 512)
    assert np.abs(got_p - want_p).max() <= 2.0 ** (3 - 23)


@pytest.mark.parametrize("w,d,u", [(14, 2, 2), (15, 1, 2)])
def test_subcircuits_of_14_and_15_wires(w, d, u):
    """The paper caps subcircuits at 15 qubits.  Above 13 wires the amplitudes of a variant live in the workspace
    instead of shared memory (same passes): a seeded HEA-shaped subcircuit against the oracle's O4/O5, whole tensor."""
    desc = hea_subcircuit(w, d, u, seed=1400 + w)
    got = tqc.tqc_simulate_subcircuit_tensor(**desc).cpu().numpy().astype(np.float64)
    sub = cutting.Subcircuit(0, w=w, gates=desc["gates"], D=[(q, i) for i, q in enumerate(desc["D_wires"])],
                             U=[(q, d + j) for j, q in enumerate(desc["U_wires"])], O=[(q, q) for q in desc["O_wires"]])
    want = cutting.build_tensor(SimpleNamespace(sub_cuts=[list(range(d + u))]), sub)
    assert got.shape == want.shape == (4 ** (d + u), 2 ** (w - u))
    assert np.abs(got - want).max() <= 2.0 ** (d - 23)
    assert abs(want[0].sum() - 2.0 ** d) < 1e-9                 # sum_x T[I...I, x] = 2^{d_s}


def test_errors():
    with pytest.raises(tqc.TqcError) as e:
        tqc.tqc_simulate_subcircuit_tensor(16, [], [], [], list(range(16)), [])
    assert e.value.code == -6
    with pytest.raises(tqc.TqcError) as e:                       # wire 1 has no end
        tqc.tqc_simulate_subcircuit_tensor(2, [], [], [0], [], [0])
    assert e.value.code == -1
    with pytest.raises(tqc.TqcError) as e:                       # wire listed twice
        tqc.tqc_simulate_subcircuit_tensor(2, [], [], [0], [0], [0])
    assert e.value.code == -1
    with pytest.raises(tqc.TqcError) as e:                       # bond_pos not a permutation
        tqc.tqc_simulate_subcircuit_tensor(2, [], [0], [1], [0], [0, 0])
    assert e.value.code == -1
    with pytest.raises(tqc.TqcError) as e:                       # two-qubit gate on one wire
        tqc.tqc_simulate_subcircuit_tensor(2, [("cz", (), (1, 1))], [], [], [0, 1], [])
    assert e.value.code == -1
    ws = torch.empty(256, dtype=torch.uint8, device="cuda")
    with pytest.raises(tqc.TqcError) as e:
        tqc.tqc_simulate_subcircuit_tensor(8, [], [0, 1], [0, 1], list(range(2, 8)), [0, 1, 2, 3], workspace=ws)
    assert e.value.code == -5
