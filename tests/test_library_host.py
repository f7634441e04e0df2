"""Host-side tests of libtqc.so — CPU only, no compute call.

* the library loads and exports every symbol include/tqc.h declares;
* the C++ planner's serialised plan is byte-identical to the oracle-side reference planner
  (rules P1-P6) on the fixtures, on random networks and on configs 3-5 —
  north_star: "bit-identical in the chosen contraction plan";
* the paper's printed multiplication counts through the library (144 / 132 / 768-bound);
* argument validation and error codes.
"""
import ctypes
import re
import os

import numpy as np
import pytest

import paper_2502_03445_b200 as tqc
from paper_2502_03445_b200 import binding
from oracle import planner_ref as P
from tqc_inputs import configs
from tqc_inputs.network import Network

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _fig5_network():
    return Network(4, [(0, 1), (1, 2), (1, 3), (2, 3)], [[0], [0, 1, 2], [1, 3], [2, 3]], [[0], [1], [2], [3]])


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "tqc.h")).read()
    declared = set(re.findall(r"\b(tqc_[a-z0-9_]+)\s*\(", header))
    declared -= {"tqc_status"}
    assert declared == set(binding.EXPORTED), declared ^ set(binding.EXPORTED)
    lib = ctypes.CDLL(tqc.lib_path())
    for name in declared:
        assert hasattr(lib, name), name
    assert "sm_100a" in tqc.version()


def test_fig5_costs_through_the_library():
    net = _fig5_network()
    p = tqc.tqc_plan(net, order=[(0, 1), (4, 2), (5, 3)])                  # the paper's order ((1,2),3),4
    assert [2 ** s["log2cost"] for s in p.steps()] == [64, 64, 16] and p.kmax == 3
    assert abs(2 ** p.cost_log2 - 144) < 1e-9
    p = tqc.tqc_plan(net, order=[(2, 3), (4, 1), (5, 0)])                  # ((3,4),2),1
    assert [2 ** s["log2cost"] for s in p.steps()] == [64, 64, 4]
    g = tqc.tqc_plan(net)
    assert 2 ** g.cost_log2 <= 144 + 1e-9 < 768                            # never worse than Fig. 5
    assert 2 ** g.cost_log2 <= net.m * 4 ** g.kmax                         # Eq. 2


def test_library_planner_against_hand_worked_step_lists():
    """The C++ planner against tests/golden/planner_steps.txt directly (not through the reference planner): operands,
    bond widths and cost exponent of every step of the three hand-worked networks."""
    from golden_planner import PLANNER_NETS, golden_planner_steps
    gold = golden_planner_steps()
    for name, make in PLANNER_NETS.items():
        p = tqc.tqc_plan(make())
        got = [(s["lhs"], s["rhs"], s["n_inner"], s["n_outer_lhs"], s["n_outer_rhs"], s["log2cost"]) for s in p.steps()]
        want = [(g["lhs"], g["rhs"], len(g["inner"]), len(g["outer_lhs"]), len(g["outer_rhs"]), g["log2cost"]) for g in gold[name]]
        assert got == want, name


@pytest.mark.parametrize("mode", [tqc.MODE_STATES, tqc.MODE_DISTRIBUTION])
def test_plan_is_bit_identical_to_reference_planner(mode):
    nets = [_fig5_network(), configs.cfg4_network()]
    if mode == tqc.MODE_STATES:
        nets.append(configs.cfg5_network())
    for seed in range(40):
        m = 2 + seed % 7
        nets.append(configs.random_network(m, m + seed % 5, 1000 + seed, connected=(seed % 4 != 0)))
    for net in nets:
        got = tqc.tqc_plan(net, mode).serialize()
        want = P.serialize(P.plan(net, mode))
        assert got == want, net.name


def test_plan_queries_and_shapes():
    net = configs.cfg4_network()
    p = tqc.tqc_plan(net)
    assert (p.n_qubits, p.m, p.K, p.num_steps, p.mode) == (64, 8, 14, 7, tqc.MODE_STATES)
    for s in range(net.m):
        assert p.tensor_shape(s) == (net.c(s), net.o(s))
    ref = P.plan(net)
    for i, st in enumerate(p.steps()):
        r = ref["steps"][i]
        assert (st["lhs"], st["rhs"], st["n_inner"], st["log2cost"]) == (r["lhs"], r["rhs"], len(r["inner"]), r["log2cost"])
    assert p.workspace_bytes(1 << 18) >= p.workspace_min_bytes() > 0
    assert p.node(2 * net.m - 2)["n_open"] == 0
    assert p.launch_count == 0


def test_degenerate_networks_plan():
    one = Network(3, [], [[]], [[2, 0, 1]])                                # K = 0, m = 1 (reading G15)
    p = tqc.tqc_plan(one, tqc.MODE_DISTRIBUTION)
    assert (p.m, p.K, p.num_steps, p.kmax) == (1, 0, 0, 0)
    disc = Network(2, [], [[], []], [[0], [1]])                            # disconnected: outer product
    p = tqc.tqc_plan(disc)
    assert p.num_steps == 1 and p.step(0)["n_inner"] == 0
    empty_out = Network(1, [(0, 1)], [[0], [0]], [[0], []])                # o_s = 0 allowed
    assert tqc.tqc_plan(empty_out).tensor_shape(1) == (1, 0)


def test_argument_errors():
    bad = Network(2, [(0, 0)], [[0], [0]], [[0], [1]])                     # cut with both ends in one subcircuit
    with pytest.raises(tqc.TqcError) as e:
        tqc.tqc_plan(bad)
    assert e.value.code == -1
    missing_q = Network(3, [(0, 1)], [[0], [0]], [[0], [1]])               # qubit 2 unowned
    with pytest.raises(tqc.TqcError):
        tqc.tqc_plan(missing_q)
    net = _fig5_network()
    with pytest.raises(tqc.TqcError):
        tqc.tqc_plan(net, order=[(0, 1), (0, 2), (5, 3)])                  # reuses a dead node
    with pytest.raises(tqc.TqcError):
        tqc.tqc_plan(net, mode=7)


def test_restarts_never_worse_and_deterministic():
    net = configs.cfg5_network()
    base = tqc.tqc_plan(net)
    a = tqc.tqc_plan(net, restarts=16, seed=7)
    b = tqc.tqc_plan(net, restarts=16, seed=7)
    assert a.serialize() == b.serialize()
    assert a.cost_log2 <= base.cost_log2 + 1e-9


def test_sliced_plan_is_the_plan_of_the_smaller_network():
    """Index slicing: the library plans the network without the sliced cuts once; its blob is
    byte-identical to the reference planner's on the oracle-side reduced network; shapes still describe the caller's tensors."""
    from oracle import reconstruct as R
    from tqc_inputs import random_tensors
    net = configs.random_network(5, 8, seed=77, o_lo=1, o_hi=3)
    T = random_tensors(net, 1)
    for slice_cuts in ([3], [0, 5], [7, 2, 4]):
        small, _ = R.slice_network(net, T, slice_cuts, [0] * len(slice_cuts))
        plan = tqc.tqc_plan(net, tqc.MODE_STATES, slice_cuts=slice_cuts, use_chain=-1)
        ref = tqc.tqc_plan(small, tqc.MODE_STATES, use_chain=-1)
        assert plan.serialize() == ref.serialize()
        assert plan.serialize() == P.serialize(P.plan(small, 0))
        assert plan.K == net.K and plan.n_sliced_cuts == len(slice_cuts)
        assert [plan.tensor_shape(s) for s in range(net.m)] == [(net.c(s), net.o(s)) for s in range(net.m)]
        assert plan.workspace_bytes(1000) >= ref.workspace_bytes(1000) + 4000
    with pytest.raises(tqc.TqcError):
        tqc.tqc_plan(net, tqc.MODE_STATES, slice_cuts=[1, 1])
    with pytest.raises(tqc.TqcError):
        tqc.tqc_plan(net, tqc.MODE_STATES, slice_cuts=[net.K])


def test_choose_slice_cuts_matches_reference_and_meets_limits():
    """Two-level slicing choice: library == oracle-side reference on random networks in both
    modes; the chosen set meets both limits (checked through the plan it leads to); infeasible limits are reported."""
    for seed in range(12):
        net = configs.random_network(3 + seed % 5, 6 + seed % 6, seed=500 + seed, o_lo=0, o_hi=4)
        for mode in (tqc.MODE_STATES, tqc.MODE_DISTRIBUTION):
            full = tqc.tqc_plan(net, mode, use_chain=-1)
            inter = max(2 * full.node(net.m + t)["n_open"] + (full.node(net.m + t)["n_bits"] if mode else 0)
                        for t in range(net.m - 1))
            big_in = max(2 * net.c(s) + net.o(s) for s in range(net.m))
            for lim_in, lim_inter in ((62, 62), (big_in - 2, 62), (62, max(inter - 3, 2)), (big_in - 3, max(inter - 4, 2))):
                want = P.choose_slice_cuts(net, mode, lim_in, lim_inter)
                if want is None:
                    with pytest.raises(tqc.TqcError):
                        tqc.tqc_choose_slice_cuts(net, mode, lim_in, lim_inter)
                    continue
                got = tqc.tqc_choose_slice_cuts(net, mode, lim_in, lim_inter)
                assert got == want, (seed, mode, lim_in, lim_inter)
                if (lim_in, lim_inter) == (62, 62):
                    assert got == []
                plan = tqc.tqc_plan(net, mode, slice_cuts=got, use_chain=-1)
                left = [net.c(s) - sum(1 for e in got if e in net.sub_cuts[s]) for s in range(net.m)]
                assert max(2 * left[s] + net.o(s) for s in range(net.m)) <= lim_in
                assert max([2 * plan.node(net.m + t)["n_open"] + (plan.node(net.m + t)["n_bits"] if mode else 0)
                            for t in range(net.m - 1)] or [0]) <= lim_inter


def test_restarts_respect_kmax_cap_and_are_deterministic():
    """Order search (PAPER.md 441-450: the role CoTenGra plays there): seeded randomised-greedy restarts keep the cheapest
    order, optionally among those whose widest step stays within kmax_cap; the same seed gives the same plan."""
    net = configs.cfg5_network()
    greedy = tqc.tqc_plan(net, tqc.MODE_STATES)
    a = tqc.tqc_plan(net, tqc.MODE_STATES, restarts=64, seed=7)
    b = tqc.tqc_plan(net, tqc.MODE_STATES, restarts=64, seed=7)
    assert a.serialize() == b.serialize()
    assert a.cost_log2 <= greedy.cost_log2 + 1e-9
    capped = tqc.tqc_plan(net, tqc.MODE_STATES, restarts=64, seed=7, kmax_cap=greedy.kmax - 1)
    assert capped.kmax <= max(greedy.kmax - 1, min(a.kmax, greedy.kmax))
    if capped.kmax <= greedy.kmax - 1:
        loose = tqc.tqc_plan(net, tqc.MODE_STATES, restarts=64, seed=7, kmax_cap=capped.kmax)
        assert loose.kmax <= capped.kmax and loose.cost_log2 <= capped.cost_log2 + 1e-9
    impossible = tqc.tqc_plan(net, tqc.MODE_STATES, restarts=16, seed=3, kmax_cap=2)      # nothing meets it: smallest K_max wins
    assert impossible.kmax <= greedy.kmax


def test_order_search_with_the_run_time_objective():
    """tqc_plan_opts.objective = 1 (host only): the search keeps the order with the smallest MODELLED run time; never worse
    than the greedy plan under that model, deterministic per seed, a valid plan (same network, m - 1 steps, root closed)."""
    net = configs.cfg5_network()
    B = configs.BATCH[5]
    greedy = tqc.tqc_plan(net, tqc.MODE_STATES, batch_hint=B)
    a = tqc.tqc_plan(net, tqc.MODE_STATES, batch_hint=B, restarts=16, seed=7, objective=1)
    b = tqc.tqc_plan(net, tqc.MODE_STATES, batch_hint=B, restarts=16, seed=7, objective=1)
    assert a.serialize() == b.serialize()
    assert 0 < a.modelled_seconds_per_state <= greedy.modelled_seconds_per_state
    assert a.num_steps == net.m - 1 and a.node(2 * net.m - 2)["n_open"] == 0
    assert tqc.tqc_plan(_fig5_network(), tqc.MODE_DISTRIBUTION).modelled_seconds_per_state < 0      # states mode only
    # finalize before the tensors are there is a state error, with no CUDA call involved
    with pytest.raises(tqc.TqcError) as ei:
        binding._check(binding._lib.tqc_plan_finalize(a._h, None))
    assert ei.value.code == -3


def test_simulate_description_checks_run_without_a_gpu():
    # tqc_simulate_subcircuit_tensor validates its description on the host before any CUDA call (include/tqc.h)
    import ctypes
    from paper_2502_03445_b200.binding import _lib, _subcircuit_desc
    gates = [("h", (), (0,)), ("rzz", (0.3,), (0, 1))]
    ws = binding.tqc_simulate_workspace_bytes(2, gates, [0], [1], [0], [1, 0])
    # gate table (272 B per gate, rounded to 256) + 4^2 * 2 float64 entries
    assert ws == 768 + 256
    assert binding.tqc_simulate_workspace_bytes(20, [], list(range(8)), list(range(8)), list(range(8, 20)), list(range(16))) == 0
    fake = ctypes.c_void_p(256)
    for bad, code in (((2, gates, [0], [0], [], [1, 0]), -1),           # u + o != w
                      ((2, [("h", (), (5,))], [], [], [0, 1], []), -1),  # gate wire out of range
                      ((16, [], [], [], list(range(16)), []), -6)):      # more than 15 wires
        desc, _keep = _subcircuit_desc(*bad)
        assert _lib.tqc_simulate_subcircuit_tensor(ctypes.byref(desc), fake, fake, 1 << 30, None) == code
    with pytest.raises(binding.TqcError):
        binding.tqc_simulate_workspace_bytes(1, [("nope", (), (0,))], [], [], [0], [])
