"""Circuit -> distribution through the library alone (GPU): tqc_plan_from_gates partitions the circuit (Alg. 2/3), every
subcircuit tensor comes from the device simulation of its variants (tqc_plan_cut_subcircuit -> tqc_simulate_subcircuit_tensor),
the plan contracts them.  Checked against the UNCUT float64 statevector (the paper's correctness claim) and against the
closed-form output laws of the GHZ / W-state families."""
import numpy as np
import pytest
import torch

import paper_2502_03445_b200 as tqc
from oracle import cutting, statevector as sv
from oracle.direct_sum_c import direct_sum_c
from tqc_inputs import circuits as C, configs, pack_states, random_states

pytestmark = pytest.mark.gpu
TOL = 1e-5


def plan_with_device_tensors(circ, w_max, s_max, mode, **kw):
    plan = tqc.tqc_plan_from_gates(circ.n, circ.gates, w_max, s_max, mode=mode, **kw)
    for s in range(plan.m):
        sub = plan.cut_subcircuit(s)
        t = tqc.tqc_simulate_subcircuit_tensor(sub["w"], sub["gates"], sub["D_wires"], sub["U_wires"], sub["O_wires"], sub["bond_pos"])
        tqc.tqc_load_subcircuit_tensors(plan, s, t)
    return plan


@pytest.mark.parametrize("name,w_max,s_max", [("cfg1", 5, 20), ("cfg2", 10, 30), ("aqft", 7, 14), ("erdos", 6, 8)])
def test_circuit_to_distribution_against_uncut_statevector(name, w_max, s_max):
    circ = {"cfg1": configs.cfg1_circuit, "cfg2": configs.cfg2_circuit, "aqft": lambda: C.aqft_circuit(10, seed=3),
            "erdos": lambda: C.qaoa_graph_circuit(8, "erdos", 11)}[name]()
    plan = plan_with_device_tensors(circ, w_max, s_max, tqc.MODE_DISTRIBUTION)
    net = plan.cut_network()
    assert net.m >= 2 and net.K >= 1
    got = tqc.tqc_contract_distribution(plan).cpu().numpy().astype(np.float64)
    want = sv.uncut_probabilities(circ.n, circ.gates)
    print(f"{name}: library partition m = {net.m}, K = {net.K}; max |dp| / max p = {np.abs(got - want).max() / want.max():.2e}")
    assert np.abs(got - want).max() <= TOL * want.max()
    assert abs(got.sum() - 1.0) < 1e-4


def test_ghz_and_wstate_output_laws():
    n = 12
    ghz = plan_with_device_tensors(C.ghz_circuit(n), 5, 4, tqc.MODE_DISTRIBUTION)
    assert ghz.cut_network().m >= 3
    p = tqc.tqc_contract_distribution(ghz).cpu().numpy().astype(np.float64)
    assert abs(p[0] - 0.5) <= TOL and abs(p[-1] - 0.5) <= TOL and np.abs(p[1:-1]).max() <= TOL          # two dominating states
    w = plan_with_device_tensors(C.wstate_circuit(n), 5, 10, tqc.MODE_DISTRIBUTION)
    assert w.cut_network().m >= 3
    q = tqc.tqc_contract_distribution(w).cpu().numpy().astype(np.float64)
    hot = [1 << k for k in range(n)]
    assert np.abs(q[hot] - 1.0 / n).max() <= TOL / n                                                     # n states x 1/n
    rest = np.delete(q, hot)
    assert np.abs(rest).max() <= TOL / n


def test_cfg3_circuit_to_states_through_the_library():
    """30 qubits: the uncut statevector is out of reach, so the values are checked against the float64 direct sum over the
    ORACLE's tensors for the library's partition (O3-O6), 4096 states."""
    circ = configs.cfg3_circuit()
    plan = plan_with_device_tensors(circ, 12, 40, tqc.MODE_STATES, batch_hint=configs.BATCH[3])
    parts = plan.cut_assignment(len(circ.gates))
    circ.parts = [parts[i] if len(qs) == 2 else None for i, (_n, _p, qs) in enumerate(circ.gates)]
    onet, T64, _ = cutting.tensors_from_circuit(circ)
    assert onet.K <= 12
    bits = random_states(30, 4096, 77)
    got = tqc.tqc_contract_states(plan, torch.from_numpy(pack_states(bits).view(np.int64)).cuda())
    torch.cuda.synchronize()
    want, _ = direct_sum_c(onet, T64, bits)
    err = np.abs(got.cpu().numpy().astype(np.float64) - want).max()
    print(f"cfg3 circuit through the library: m = {onet.m}, K = {onet.K}, max |dp| / max p = {err / want.max():.2e}")
    assert err <= TOL * want.max()
