"""bench.py — states/s of the reconstruction hot path on B200 (one JSON line on rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4|cfg5|cfg3|cfg2] [--impl reference]

A step is ONE pass of the whole hot path (a2 key extraction, a3 gather, a4 pairwise
contractions, a5 final reduction — or a6 for a distribution workload) over one batch of
seeded synthetic input, through the C ABI (include/tqc.h).  `value` = states / s with the batch
resident in HBM; `e2e` = the same through tqc_contract_*_host with pinned HOST buffers (H2D of
the states and D2H of the probabilities inside the timed region).  Multi-GPU (torchrun): the
path shards over independent states; every rank holds the tensors and
contracts its own seeded batch, no collective on the data path ("scaling": "weak").

`--impl reference` times the CPU oracle (oracle/, float64 direct sum / per-state tensordot contraction) on a
bounded sample of the same workload; the `cpu_baseline` leg of the default arm does the same
once.  These two legs are the only places this file touches oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "reconstructed output-state probabilities/sec"
UNIT = "states/s"
SM_COUNT = 148                  # B200 (B200_PROFILING.md)
FP32_LANES_PER_SM = 128
NOMINAL_TF32_OVER_BF16 = 1.1 / 2.25   # nominal dense peaks (B200_PROFILING.md table)
TC_KERNEL_NAMES = "step_tc2_kernel on CTA pairs, step_tc_kernel<BN> on one CTA"


def measured_peaks() -> dict:
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        p["source"] = "measured"
        return p
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0,
            "source": "fallback"}


def roof_peaks() -> dict:
    """Every roofline denominator with its source.  HBM and bf16 come from MEASURED_PEAKS.json (driver-written); TF32
    matmul, FP32 FFMA, shared-memory LDS.128 and L2 read rates from profiles/peaks_r02.json, written on a B200 of this
    pool by `python -m paper_2502_03445_b200.measure_peaks` (measured by the build).  Where that file
    is missing the value is DERIVED from unit counts x sm_max_mhz (FFMA, LDS) or from bf16 x the nominal ratio (TF32)
    and labelled so."""
    p = measured_peaks()
    own_path = os.path.join(ROOT, "profiles", "peaks_r02.json")
    own = {}
    if os.path.exists(own_path):
        with open(own_path) as f:
            own = json.load(f)
    mhz = p.get("sm_max_mhz", 1965.0)
    out = dict(p)
    def pick(key, derived, how):
        if key in own:
            out[key], out[key + "_source"] = float(own[key]), "measured (profiles/peaks_r02.json)"
        else:
            out[key], out[key + "_source"] = derived, "derived: " + how
    pick("tf32_tflops", p["bf16_tflops"] * NOMINAL_TF32_OVER_BF16, "bf16 x nominal tf32/bf16 ratio 1.1/2.25")
    pick("tf32_tflops_sustained", p.get("bf16_tflops_sustained", p["bf16_tflops"]) * NOMINAL_TF32_OVER_BF16,
         "sustained bf16 x nominal tf32/bf16 ratio")
    pick("ffma_tflops", SM_COUNT * FP32_LANES_PER_SM * 2 * mhz * 1e6 / 1e12, "148 SMs x 128 lanes x 2 x sm_max_mhz")
    pick("lds_gbs", SM_COUNT * 128 * mhz * 1e6 / 1e9, "148 SMs x 128 B/clk x sm_max_mhz")
    pick("l2_read_gbs", None, "not measured")
    return out


# ---------------------------------------------------------------------------------------------
# workloads: the BASELINE.json configs as seeded synthetic inputs (tqc_inputs/, DESIGN.md recipe)
# ---------------------------------------------------------------------------------------------
def make_workload(name: str, batch: int | None = None):
    from tqc_inputs import configs, random_tensors, seed_for
    from tqc_inputs.network import Network
    from tqc_inputs.seeds import STREAM_TENSORS
    if name == "cfg4":
        net, cfg = configs.cfg4_network(), 4
    elif name == "cfg5":
        net, cfg = configs.cfg5_network(), 5
    elif name == "cfg3":
        # network shape of cfg3 (30-qubit ansatz, K = 6, tensors (3,10) (6,9) (3,11)); for timing the tensor VALUES
        # are seeded random (the statevector-simulated ones are oracle output and are used by the parity tests)
        net = Network(30, [(0, 1), (1, 0), (0, 1), (1, 2), (2, 1), (1, 2)], [[0, 1, 2], [0, 1, 2, 3, 4, 5], [3, 4, 5]],
                      [list(range(0, 10)), list(range(10, 19)), list(range(19, 30))], name="cfg3-shape")
        net.validate()
        cfg = 3
    elif name == "cfg2":
        # the cut network the seeded cfg2 circuit yields (20 qubits, 3 subcircuits, K = 5; tests/test_gpu_configs.py
        # derives it from the circuit), distribution mode, random values for timing
        net = Network(20, [(0, 1), (1, 2), (0, 2), (0, 2), (1, 2)], [[0, 2, 3], [0, 1, 4], [1, 2, 3, 4]],
                      [[0, 7, 10], [1, 2, 3, 11, 13, 17, 18, 19], [4, 5, 6, 8, 9, 12, 14, 15, 16]], name="cfg2-shape")
        net.validate()
        cfg = 2
    else:
        raise SystemExit(f"unknown workload {name}")
    B = batch if batch else configs.BATCH[cfg]
    tensors = random_tensors(net, seed_for(cfg, STREAM_TENSORS))
    return {"name": name, "cfg": cfg, "net": net, "tensors": tensors, "mode": configs.MODE[cfg], "B": int(B),
            "full_B": configs.BATCH[cfg]}


def pack_states_of(wl, rank: int, world: int = 1) -> np.ndarray:
    from tqc_inputs import pack_states
    return pack_states(workload_states(wl, rank, world)).view(np.int64)


def workload_states(wl, rank: int, world: int = 1) -> np.ndarray:
    """(B, n) bits of THIS rank: the job's batch is the first world x B states of the config's seeded batch (uniform over
    {0,1}^n), cut into contiguous per-rank ranges by paper_2502_03445_b200.sharding.shard_states (states
    shard across ranks, tensors are replicated, no collective on the data path).  Weak scaling: B states per GPU."""
    from paper_2502_03445_b200.sharding import shard_states
    from tqc_inputs import random_states, seed_for
    from tqc_inputs.seeds import STREAM_STATES
    full = random_states(wl["net"].n_qubits, wl["B"] * world, seed_for(wl["cfg"], STREAM_STATES))
    lo, hi = shard_states(wl["B"] * world, rank, world)
    return full[lo:hi]


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 20 ms while the timed regions run."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                                          "-lms", "20", "-i", str(index)], stdout=self.tmp, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None
        t0 = time.time()
        while self.proc is not None and time.time() - t0 < 3.0 and os.path.getsize(self.tmp.name) == 0:
            time.sleep(0.02)                                            # first sample before the timed region starts

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.tmp.flush()
        self.tmp.seek(0)
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.tmp.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        self.tmp.close()
        os.unlink(self.tmp.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        # samples under load: the upper half of the clock readings (idle samples sit at the floor clock)
        load = sorted(sm)[len(sm) // 2:]
        return {"sm_mhz": float(np.median(load)), "sm_max_mhz": float(max(smax)), "samples": len(sm),
                "power_w_max": float(max(power)), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------
# algorithmic work of one plan step
# ---------------------------------------------------------------------------------------------
def step_work(plan, t: int, B: int, mode_states: bool):
    """(flop, bytes) one launch of plan step t must do.  flop = 2 x the paper's multiplication count
    4^{#inner+#outer} x rows; bytes = compulsory operand reads + result write, fp32."""
    NODE_BATCH = 2
    st = plan.step(t)
    m = plan.m
    c_node = plan.node(m + t)
    if mode_states:
        rows = B if c_node["kind"] == NODE_BATCH else (1 << c_node["n_bits"])
        flop = 2.0 * (2.0 ** st["log2cost"]) * rows
    else:
        rows = 1 << c_node["n_bits"]
        flop = 2.0 * (2.0 ** st["log2cost"])
    nbytes = 4.0 * rows * (4.0 ** c_node["n_open"])
    for v in (st["lhs"], st["rhs"]):
        nd = plan.node(v)
        distinct = min(rows, 1 << nd["n_bits"]) if nd["kind"] != NODE_BATCH else rows
        nbytes += 4.0 * distinct * (4.0 ** nd["n_open"])
    return flop, nbytes


def roofline_for(plan, tag: int, avg_ms: float, B: int, mode_states: bool, peaks: dict, traffic, long_step: bool = False):
    """Roofline object for the dominant launch (tag = plan step index)."""
    if tag == -4 and avg_ms > 0:
        # fused chain kernel: every per-state step of the plan in one launch
        NODE_BATCH = 2
        flop, nbytes, seen = 0.0, 4.0 * B, set()
        for t in range(plan.num_steps):
            st = plan.step(t)
            if st["kernel_class"] != 3:
                continue
            flop += 2.0 * (2.0 ** st["log2cost"]) * B
            for v in (st["lhs"], st["rhs"]):
                nd = plan.node(v)
                if nd["kind"] != NODE_BATCH and v not in seen:          # gathered operand: distinct slices once + its keys
                    seen.add(v)
                    nbytes += 4.0 * min(B, 1 << nd["n_bits"]) * (4.0 ** nd["n_open"]) + 4.0 * B
        alu_peak = peaks["ffma_tflops"]
        sec = avg_ms * 1e-3
        t_alu, t_hbm = flop / (alu_peak * 1e12), nbytes / (peaks["hbm_gbs"] * 1e9)
        if t_hbm > t_alu:
            bound, peak, unit, achieved = "hbm", peaks["hbm_gbs"], "GB/s", nbytes / sec / 1e9
        else:
            bound, peak, unit, achieved = "alu", alu_peak, "TFLOP/s", flop / sec / 1e12
        return {"bound": bound, "achieved": achieved, "peak": peak, "unit": unit, "frac": achieved / peak,
                "traffic": traffic, "kernel": "chain_spec_kernel / chain_kernel (fused per-state chain: fp32 FFMA steps + 3xTF32 mma.sync blocks for 16x16x16-class steps; specialised per plan when NVRTC is present; the FP32-ALU peak is the reference for its algorithmic flops)", "plan_step": "all per-state steps",
                "algorithmic_flop": flop, "algorithmic_bytes": nbytes, "avg_launch_ms": avg_ms,
                "peak_source": (peaks["source"] + " hbm copy") if bound == "hbm" else ("FP32 FFMA rate, " + peaks["ffma_tflops_source"])}
    if tag < 0 or avg_ms <= 0:
        return {"bound": "hbm", "achieved": None, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": None,
                "traffic": traffic, "kernel": {-1: "key_kernel", -2: "gather_kernel"}.get(tag, "?")}
    flop, nbytes = step_work(plan, tag, B, mode_states)
    kclass = plan.step(tag)["kernel_class"]
    alu_peak = peaks["ffma_tflops"]                    # TFLOP/s fp32 FFMA
    # a tensor-pipe launch inside a seconds-long cfg5 step runs under the power cap: the sustained matmul figure
    tf32_peak = peaks["tf32_tflops_sustained"] if long_step else peaks["tf32_tflops"]
    t_hbm = nbytes / (peaks["hbm_gbs"] * 1e9)
    sec = avg_ms * 1e-3
    name = {0: "step_tile_kernel (fp32 FFMA)", 1: "dot_kernel", 2: "tensor-pipe step kernel (3xTF32 tcgen05: " + TC_KERNEL_NAMES + ")"}.get(kclass, "?")
    st_ = plan.step(tag)
    if kclass == 0 and (not mode_states or plan.node(plan.m + tag)["kind"] == 1):
        # cross-mode step: the launcher's integer rule for the warp-level tensor-core tile kernel
        la, lb = plan.node(st_["lhs"]), plan.node(st_["rhs"])
        lgm = la["n_bits"] + 2 * st_["n_outer_lhs"]
        lgn = lb["n_bits"] + 2 * st_["n_outer_rhs"]
        if 3 <= 2 * st_["n_inner"] <= 6 and min(lgm, lgn) >= 6 and max(lgm, lgn) >= 7:
            name = "cross_mma_kernel (3xTF32 mma.sync tiles; FP32-ALU peak as reference)"
    if kclass == 2:
        t_cmp, peak, unit, bound = 3.0 * flop / (tf32_peak * 1e12), tf32_peak, "TFLOP/s", "tensor"
        achieved = 3.0 * flop / sec / 1e12            # issued tensor flops: 3 TF32 MMAs per fp32-accurate product
    else:
        t_cmp, peak, unit, bound = flop / (alu_peak * 1e12), alu_peak, "TFLOP/s", "alu"
        achieved = flop / sec / 1e12
    if t_hbm > t_cmp:
        bound, peak, unit, achieved = "hbm", peaks["hbm_gbs"], "GB/s", nbytes / sec / 1e9
    src = (peaks["source"] + " hbm copy") if bound == "hbm" else ("FP32 FFMA rate, " + peaks["ffma_tflops_source"]) if bound == "alu" \
        else (("sustained " if long_step else "burst ") + "TF32 matmul, " + peaks["tf32_tflops_source"])
    roof = {"bound": bound, "achieved": achieved, "peak": peak, "unit": unit, "frac": achieved / peak,
            "traffic": traffic, "kernel": name, "plan_step": tag, "algorithmic_flop": flop, "algorithmic_bytes": nbytes,
            "avg_launch_ms": avg_ms, "peak_source": src}
    if bound == "tensor":
        # both denominators SURVEY H1 asks for: issued 3xTF32 flops against the TF32 peak (frac), and the fp32-equivalent
        # rate against TF32 / 3
        roof["fp32_equivalent_tflops"] = flop / sec / 1e12
        roof["frac_of_tf32_over_3"] = (flop / sec / 1e12) / (tf32_peak / 3.0)
    return roof


def committed_traffic(workload: str, tag: int, states_per_launch: float):
    """DRAM bytes per launch of the dominant kernel (dram__bytes_read.sum + dram__bytes_write.sum) from the committed
    `ncu --set full` captures listed in profiles/traffic.csv, scaled to this run's states per launch; else None."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path):
        return None
    with open(path) as f:
        for line in f.read().splitlines()[1:]:
            parts = line.split(",")
            if len(parts) >= 4 and parts[0] == workload and parts[1] == str(tag):
                return float(parts[3]) * states_per_launch / float(parts[2])
    return None


# ---------------------------------------------------------------------------------------------
# the GPU arm
# ---------------------------------------------------------------------------------------------
def run_ours(args) -> None:
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    import paper_2502_03445_b200 as tqc      # fails loudly if libtqc.so is missing

    ctx = {"torch": torch, "dist": dist, "tqc": tqc, "world": world, "rank": rank, "local": local, "dev": dev}
    if args.workload == "variants":
        if rank == 0:
            print(json.dumps(measure_variants(ctx, args.steps, args.warmup, not args.no_cpu_baseline)), flush=True)
        if world > 1:
            dist.destroy_process_group()
        return
    # cfg5 without --batch: the 8d-5 prefix rule (batch = -1); --batch N times the first N states; --batch 1000000 the full batch
    head_batch = args.batch if args.batch > 0 else (-1 if args.workload == "cfg5" else 0)
    line = measure(ctx, args, args.workload, head_batch, args.steps, args.warmup)
    if rank == 0:
        if world == 1 and args.others:
            # the other BASELINE configs, shorter runs, same protocol (cfg5: a labelled prefix of its 10^6-state batch)
            others = []
            for name, batch, steps in (("cfg5", -1, 3), ("cfg4", 0, 20), ("cfg3", 0, 10), ("cfg2", 0, 10)):
                if name == args.workload:
                    continue
                o = measure(ctx, args, name, batch, steps, 3)
                others.append({k: o[k] for k in ("value", "unit", "ms_per_step", "steps", "gpu_launches", "roofline")} |
                              {"workload": o["config"]["workload"], "e2e_value": o["e2e"]["value"],
                               "chain_status": o["config"]["chain_status"], "kernel_classes": o["config"]["kernel_classes"]})
            others.append(measure_hss(ctx, 10, 3))
            others.append(measure_hss_contract(ctx, 10, 3))
            others.append(measure_variants(ctx, 10, 3, not args.no_cpu_baseline))
            line["other_workloads"] = others
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(make_workload(args.workload, args.batch if args.batch > 0 else None), args.cpu_seconds)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def measure(ctx, args, workload: str, batch: int, steps: int, warmup: int):
    """One workload through the full protocol; returns the JSON line as a dict (rank 0) or None."""
    torch, dist, tqc = ctx["torch"], ctx["dist"], ctx["tqc"]
    world, rank, local, dev = ctx["world"], ctx["rank"], ctx["local"], ctx["dev"]
    peaks = roof_peaks()
    wl = make_workload(workload, batch if batch > 0 else None)
    net = wl["net"]
    states_mode = wl["mode"] == "states"
    # cfg5: the order search with the run-time objective (seeded restarts + tree rotations, about 15 s of host time, outside
    # every timed region); the other configs keep the deterministic greedy plan (their plans are a handful of steps)
    restarts = args.restarts if args.restarts >= 0 else (1024 if wl_name_is_cfg5(workload) else 0)
    # batch_hint = the config's FULL batch: a prefix run keeps the plan (tables, kernel classes) of the real workload
    table_log2 = args.table_log2 if args.table_log2 >= 0 else (30 if wl_name_is_cfg5(workload) else 0)
    plan = tqc.tqc_plan(net, tqc.MODE_STATES if states_mode else tqc.MODE_DISTRIBUTION, batch_hint=wl["full_B"],
                        restarts=restarts, seed=args.plan_seed, objective=1 if (restarts > 0 and states_mode) else 0,
                        table_log2_floats_max=table_log2)
    for s, t in enumerate(wl["tensors"]):
        tqc.tqc_load_subcircuit_tensors(plan, s, t)
    prefix_note = None
    if batch < 0:
        # the full batch does not fit a bench step; time a power-of-two PREFIX of the same seeded batch, the
        # smallest one whose step runs >= 1 s, found from a calibration run of 2^10 states (all ranks agree on it)
        n_cal = 1 << 10
        wl["B"] = n_cal
        cal_states = torch.from_numpy(pack_states_of(wl, rank, world)).to(dev)
        cal_ws = torch.empty(min(plan.workspace_bytes(n_cal), args.max_workspace_gb << 30), dtype=torch.uint8, device=dev)
        cal_out = torch.empty(n_cal, dtype=torch.float32, device=dev)
        for _ in range(2):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            tqc.tqc_contract_states(plan, cal_states, out=cal_out, workspace=cal_ws)
            e1.record()
            torch.cuda.synchronize()
        t_cal = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t_cal, op=dist.ReduceOp.MAX)
        lg = 10
        while (1 << lg) < wl["full_B"] and float(t_cal.item()) * (1 << (lg - 10)) < 1000.0:
            lg += 1
        wl["B"] = min(1 << lg, wl["full_B"])
        prefix_note = (f"calibration: 2^10 states in {float(t_cal.item()):.1f} ms -> smallest power-of-two prefix with a step >= 1 s "
                       f"is 2^{lg}")
        del cal_states, cal_ws, cal_out
        torch.cuda.empty_cache()
    B = wl["B"]
    n_out = B if states_mode else (1 << net.n_qubits)

    if states_mode:
        packed = pack_states_of(wl, rank, world)
        states_host = torch.from_numpy(packed).pin_memory()
        states_dev = states_host.to(dev)
        ws_bytes = min(plan.workspace_bytes_host(B), max(args.max_workspace_gb << 30,
                                                          plan.workspace_min_bytes() + (B * (packed.shape[1] * 8 + 4)) + 4096))
    else:
        states_host = states_dev = None
        ws_bytes = plan.workspace_bytes_host(0, 0)
    workspace = torch.empty(max(ws_bytes, 256), dtype=torch.uint8, device=dev)
    out_dev = torch.empty(n_out, dtype=torch.float32, device=dev)
    out_host = torch.empty(n_out, dtype=torch.float32).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2
    stream = torch.cuda.current_stream()

    def step_device():
        if states_mode:
            tqc.tqc_contract_states(plan, states_dev, out=out_dev, workspace=workspace, stream=stream)
        else:
            tqc.tqc_contract_distribution(plan, out=out_dev, workspace=workspace, stream=stream)

    def step_host():
        if states_mode:
            tqc.tqc_contract_states_host(plan, states_host, out_host, workspace, stream=stream)
        else:
            tqc.tqc_contract_distribution_host(plan, out_host, workspace, stream=stream)

    def timed(fn, steps, warmup):
        for _ in range(warmup):
            flush.zero_()
            fn()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        l0 = plan.launch_count
        for a, b in evs:
            flush.zero_()                      # L2 flush between timed iterations (outside the event pair)
            a.record(stream)
            fn()
            b.record(stream)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        ms = sum(a.elapsed_time(b) for a, b in evs)
        t = torch.tensor([ms], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item()), plan.launch_count - l0

    sampler = ClockSampler(local) if rank == 0 else None
    total_ms, launches = timed(step_device, steps, warmup)
    e2e_ms, _ = timed(step_host, steps, warmup)

    # per-launch times of the same step, CUDA events on the launching stream inside the library
    plan.profile_enable(True)
    per_tag: dict = {}
    prof_steps = steps if ms_hint_short(total_ms, steps) else min(steps, 2)
    for _ in range(prof_steps):
        flush.zero_()
        step_device()
        for tag, ms in plan.profile_read():
            acc = per_tag.setdefault(tag, [0.0, 0])
            acc[0] += ms
            acc[1] += 1
    plan.profile_enable(False)
    torch.cuda.synchronize()
    clocks = sampler.stop() if sampler else None

    chain_rc, chain_note = plan.chain_status()
    ms_per_step = total_ms / steps
    value = world * n_out / (ms_per_step * 1e-3)
    e2e_value = world * n_out / (e2e_ms / steps * 1e-3)
    if rank != 0:
        return None

    dom = max(per_tag.items(), key=lambda kv: kv[1][0])
    dom_tag, (dom_total, dom_n) = dom
    launches_per_step = dom_n / prof_steps
    rows_B = B / launches_per_step if states_mode else B          # a chunked batch runs the step once per chunk
    roof = roofline_for(plan, dom_tag, dom_total / dom_n, int(rows_B), states_mode, peaks,
                        committed_traffic(wl["name"], dom_tag, rows_B), long_step=ms_per_step > 200.0)
    step_ms_sum = sum(v[0] for v in per_tag.values()) / prof_steps
    roof["share_of_step"] = (dom_total / prof_steps) / step_ms_sum if step_ms_sum > 0 else None
    kclass_name = {0: "simt_tile", 1: "dot", 2: "tcgen05", 3: "chain"}
    kernels = {}
    for tag, v in sorted(per_tag.items()):
        ent = {"ms_per_step": v[0] / prof_steps, "launches_per_step": v[1] / prof_steps}
        if tag >= 0:
            st_ = plan.step(tag)
            ent["kernel_class"] = kclass_name.get(st_["kernel_class"], "?")
            ent["log2_mults_per_row"] = st_["log2cost"]
        else:
            ent["kernel_class"] = {-1: "key_kernel", -2: "gather_kernel", -4: "fused chain"}.get(tag, "?")
        kernels[str(tag)] = ent
    # whole-step tensor-pipe accounting (cfg5): algorithmic flops of every tcgen05 step over their summed launch time
    tc_flop = sum(2.0 * 2.0 ** plan.step(t)["log2cost"] * B for t in range(plan.num_steps) if plan.step(t)["kernel_class"] == 2)
    tc_ms = sum(v[0] / prof_steps for tag, v in per_tag.items() if tag >= 0 and plan.step(tag)["kernel_class"] == 2)
    if tc_ms > 0:
        tfs = tc_flop / (tc_ms * 1e-3) / 1e12
        pk = peaks["tf32_tflops_sustained"] if ms_per_step > 200.0 else peaks["tf32_tflops"]
        roof["all_tensor_steps"] = {"fp32_equivalent_tflops": tfs, "ms_per_step": tc_ms, "frac_of_tf32_over_3": tfs / (pk / 3.0),
                                    "frac_of_tf32_issued": 3.0 * tfs / pk}

    words = (net.n_qubits + 63) // 64
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_description(wl, plan), "states_per_step_per_gpu": n_out,
                   "parallelism": f"states sharded over {world} GPU(s), tensors replicated, no collective",
                   "l2": "flushed between timed iterations (256 MB write)", "plan_cost_log2_per_state": plan.cost_log2, "planner_restarts": restarts, "table_log2_floats_max": table_log2 or 24,
                   "planner_objective": "modelled run time (tqc_plan_opts.objective = 1)" if (restarts > 0 and states_mode) else "deterministic greedy",
                   "planner_modelled_us_per_state": plan.modelled_seconds_per_state * 1e6 if states_mode else None,
                   "kmax": plan.kmax, "workspace_gb": ws_bytes / 2 ** 30, "prefix_rule": prefix_note,
                   "library": tqc.version(), "chain_status": chain_rc, "chain_note": chain_note,
                   "kernel_classes": {kclass_name[k]: sum(1 for t in range(plan.num_steps) if plan.step(t)["kernel_class"] == k)
                                      for k in kclass_name}},
        "e2e": {"value": e2e_value, "unit": UNIT,
                "h2d_bytes_per_step": int(B * words * 8) if states_mode else 0, "d2h_bytes_per_step": int(n_out * 4)},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": roof,
        "kernels_ms": kernels,
    }
    plan.close()
    del workspace, flush, out_dev
    torch.cuda.empty_cache()
    return line


def wl_name_is_cfg5(name: str) -> bool:
    return name == "cfg5"


def ms_hint_short(total_ms: float, steps: int) -> bool:
    """True when a step is short enough to repeat the per-launch profiling pass `steps` times."""
    return total_ms / max(steps, 1) < 50.0


def measure_hss(ctx, steps: int, warmup: int) -> dict:
    """NEXT row 1 (Alg. 1): the state-norm pass over two 4^6 x 2^14 tensors (512 MB, larger than L2), one launch
    per subcircuit, against the HBM copy peak.  Selection and expansion are host work and are not timed here."""
    torch, tqc, dev = ctx["torch"], ctx["tqc"], ctx["dev"]
    from tqc_inputs.network import Network
    K, o = 6, 14
    net = Network(2 * o, [(0, 1)] * K, [list(range(K)), list(range(K))], [list(range(o)), list(range(o, 2 * o))],
                  name="hss-2x(4^6 x 2^14)")
    net.validate()
    plan = tqc.tqc_plan(net, tqc.MODE_STATES)
    rng = np.random.default_rng(250203445)
    for s in range(net.m):
        tqc.tqc_load_subcircuit_tensors(plan, s, rng.random((4 ** K, 2 ** o), dtype=np.float32))
    scores = [torch.empty(2 ** o, dtype=torch.float32, device=dev) for _ in range(net.m)]
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    l0 = plan.launch_count
    for _ in range(warmup):
        for s in range(net.m):
            tqc.tqc_hss_scores(plan, s, out=scores[s], stream=stream)
    torch.cuda.synchronize()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in evs:
        flush.zero_()
        a.record(stream)
        for s in range(net.m):
            tqc.tqc_hss_scores(plan, s, out=scores[s], stream=stream)
        b.record(stream)
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in evs) / steps
    nbytes = net.m * (4 ** K * 2 ** o + 2 ** o) * 4
    peaks = roof_peaks()
    gbs = nbytes / (ms * 1e-3) / 1e9
    launches = plan.launch_count - l0
    plan.close()
    return {"workload": f"{net.name}: tqc_hss_scores over both subcircuits", "value": net.m * 2 ** o / (ms * 1e-3),
            "unit": "subcircuit states scored/s", "ms_per_step": ms, "steps": steps, "gpu_launches": int(launches),
            "roofline": {"bound": "hbm", "kernel": "hss_norm_kernel<32>", "achieved": gbs, "peak": peaks["hbm_gbs"],
                         "unit": "GB/s", "frac": gbs / peaks["hbm_gbs"], "traffic": None, "peak_source": peaks["source"],
                         "algorithmic_bytes_per_launch": nbytes // net.m}}


def measure_variants(ctx, steps: int, warmup: int, with_cpu: bool = True) -> dict:
    """NEXT row 4 (section 2.1): T_s of one subcircuit from a device simulation of its 4^d 3^u variants.  Synthetic
    subcircuit with the shape of cfg3's middle one (12 wires, d = u = 3, o = 9; three RY/RZ layers, two CX ladders, seeded
    angles): 1728 variants, one block each.  The amplitudes never leave shared memory, so the bound is the shared-memory
    pipe: every pass reads and writes the 2^w amplitudes once (peak = 148 SMs x 128 B/clk x sm_max_mhz)."""
    torch, tqc, dev = ctx["torch"], ctx["tqc"], ctx["dev"]
    from tqc_inputs.circuits import hea_subcircuit
    w, d, u = 12, 3, 3
    desc = hea_subcircuit(w, d, u)
    gates = desc["gates"]
    out = torch.empty((4 ** (d + u), 2 ** (w - u)), dtype=torch.float32, device=dev)
    ws = torch.empty(tqc.tqc_simulate_workspace_bytes(**desc), dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    for _ in range(warmup):
        tqc.tqc_simulate_subcircuit_tensor(**desc, out=out, workspace=ws, stream=stream)
    torch.cuda.synchronize()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in evs:
        flush.zero_()
        a.record(stream)
        tqc.tqc_simulate_subcircuit_tensor(**desc, out=out, workspace=ws, stream=stream)
        b.record(stream)
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in evs) / steps
    variants = 4 ** d * 3 ** u
    peaks = roof_peaks()
    # Algorithmic shared-memory bytes: per preparation one pass per two-qubit gate (the one-qubit gates are
    # folded into them on the host), 32 B per amplitude (complex128 read + write); per setting one rotation pass (32 B),
    # |amp|^2 (16 B read + 8 B write), u Walsh-Hadamard passes over float64 (16 B each) and the scatter read (8 B).
    n2q = sum(1 for g in gates if len(g[2]) == 2)
    smem_bytes = 4 ** d * 2 ** w * (n2q * 32 + 3 ** u * (32 + 24 + 16 * u + 8))
    # what the launch issues: the library splits the 3^u settings of a preparation over 3^g blocks (g = 2 here: 576
    # blocks, two per SM) and each of them repeats the preparation's gate passes
    g_fixed, blocks = 0, 4 ** d
    while g_fixed < u and blocks < 2 * 148:
        blocks, g_fixed = blocks * 3, g_fixed + 1
    issued_bytes = 2 ** w * (blocks * (n2q + 2.0 * g_fixed / 3.0) * 32 + 4 ** d * 3 ** u * (24 + 16 * u + 8)
                             + (4 ** d * 3 ** u - blocks) * 32)
    peak = peaks["lds_gbs"]                                    # measured LDS.128 rate (profiles/peaks_r02.json), else derived
    gbs = smem_bytes / (ms * 1e-3) / 1e9
    assert abs(float(out[0].sum()) - 2 ** d) < 1e-3                # sum_x T[I...I, x] = 2^{d_s} (reading G16)
    cpu = None
    if with_cpu:
        # the oracle as it stands (O4/O5, numpy float64, one thread) on the SAME subcircuit, whole tensor; also a parity
        # check of the timed configuration: |dT| <= 2^d 2^-23
        from oracle import cutting
        from types import SimpleNamespace
        sub = cutting.Subcircuit(0, w=w, gates=gates, D=[(q, i) for i, q in enumerate(desc["D_wires"])],
                                 U=[(q, d + j) for j, q in enumerate(desc["U_wires"])],
                                 O=[(q, q) for q in desc["O_wires"]])
        net1 = SimpleNamespace(sub_cuts=[list(range(d + u))])     # build_tensor reads only the subcircuit's axis order
        t0 = time.perf_counter()
        want = cutting.build_tensor(net1, sub)
        sec = time.perf_counter() - t0
        err = float(np.abs(out.cpu().numpy().astype(np.float64) - want).max())
        assert err <= 2.0 ** (d - 23), ("variants row against the oracle", err)
        cpu = {"value": variants / sec, "unit": "subcircuit variants simulated/s", "cores": 1, "kind": "oracle",
               "sample": f"oracle.cutting.build_tensor on the same subcircuit, all {variants} variants, {sec:.1f} s; "
                         f"max |T_gpu - T_oracle| = {err:.2e}"}
    return {"workload": f"variants: {w}-wire subcircuit, d = u = 3, {len(gates)} gates, {variants} variants -> T_s "
                        f"[4^6][2^9] (tqc_simulate_subcircuit_tensor)",
            "value": variants / (ms * 1e-3), "unit": "subcircuit variants simulated/s", "ms_per_step": ms, "steps": steps,
            "gpu_launches": 2 + d,
            "roofline": {"bound": "smem", "kernel": "sim_variant_kernel (whole call timed: + 3 sim_kappa_axis_kernel + "
                                                    "sim_permute_cast_kernel)",
                         "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "traffic": None,
                         "peak_source": "shared-memory LDS.128 rate, " + peaks["lds_gbs_source"],
                         "algorithmic_bytes_per_launch": smem_bytes, "issued_bytes_per_launch": issued_bytes,
                         "issued_gbs": issued_bytes / (ms * 1e-3) / 1e9},
            "cpu_baseline": cpu}


def measure_hss_contract(ctx, steps: int, warmup: int) -> dict:
    """NEXT row 1, pruned contraction: Alg. 1 selection of >= 2^20 composite states on the cfg3-shaped network, contracted
    once with pruned output axes (tqc_hss_contract) and, for comparison, state by state (tqc_contract_states on the
    expanded batch).  A step = scores + (host) selection excluded; prepare + contract timed."""
    torch, tqc, dev = ctx["torch"], ctx["tqc"], ctx["dev"]
    wl = make_workload("cfg3")
    net = wl["net"]
    plan = tqc.tqc_plan(net, tqc.MODE_STATES, batch_hint=1 << 20)
    for s, t in enumerate(wl["tensors"]):
        tqc.tqc_load_subcircuit_tensors(plan, s, t)
    scores = [tqc.tqc_hss_scores(plan, s) for s in range(net.m)]
    torch.cuda.synchronize()
    x = tqc.tqc_hss_select(plan, [v.cpu().numpy() for v in scores], 1 << 20)
    n = int(np.prod([len(v) for v in x], dtype=np.int64))
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    out = torch.empty(n, dtype=torch.float32, device=dev)
    l0 = plan.launch_count

    def timed(fn):
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in evs:
            flush.zero_()
            a.record(stream)
            fn()
            b.record(stream)
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in evs) / steps

    ms_product = timed(lambda: tqc.tqc_hss_contract(plan, x, out=out, stream=stream))
    launches = (plan.launch_count - l0) // (steps + warmup)
    states = torch.from_numpy(tqc.tqc_hss_expand(plan, x).view(np.int64)).to(dev)
    ws = torch.empty(plan.workspace_bytes(n), dtype=torch.uint8, device=dev)
    out2 = torch.empty(n, dtype=torch.float32, device=dev)
    ms_states = timed(lambda: tqc.tqc_contract_states(plan, states, out=out2, workspace=ws, stream=stream))
    torch.cuda.synchronize()
    agree = float((out - out2).abs().max() / out2.abs().max())
    # algorithmic work of the pruned contraction: 2 x the multiplication count of its plan (tqc_hss_cost_log2) against the
    # measured FFMA rate; bytes = the pruned tensors read once + the result written once
    peaks = roof_peaks()
    flop = 2.0 * 2.0 ** plan.hss_cost_log2
    nbytes = 4.0 * (sum(len(v) * 4.0 ** len(net.sub_cuts[j]) for j, v in enumerate(x)) + n)
    sec = ms_product * 1e-3
    t_alu, t_hbm = flop / (peaks["ffma_tflops"] * 1e12), nbytes / (peaks["hbm_gbs"] * 1e9)
    if t_alu >= t_hbm:
        roof = {"bound": "alu", "achieved": flop / sec / 1e12, "peak": peaks["ffma_tflops"], "unit": "TFLOP/s",
                "peak_source": "FP32 FFMA rate, " + peaks["ffma_tflops_source"]}
    else:
        roof = {"bound": "hbm", "achieved": nbytes / sec / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "peak_source": peaks["source"] + " hbm copy"}
    roof.update({"frac": roof["achieved"] / roof["peak"], "traffic": None, "algorithmic_flop": flop, "algorithmic_bytes": nbytes,
                 "kernel": "whole call: hss_rows_kernel (pruned tensors) + distribution-mode steps (step_tile / cross_mma) + hss_compact_kernel"})
    plan.close()
    return {"workload": f"hss-contract: cfg3-shaped network, |x_j| = {[len(v) for v in x]}, {n} composite states",
            "value": n / (ms_product * 1e-3), "unit": UNIT, "ms_per_step": ms_product, "steps": steps,
            "gpu_launches": int(launches), "per_state_path_ms": ms_states, "max_rel_diff_vs_per_state_path": agree,
            "roofline": roof}


def workload_description(wl, plan) -> str:
    net = wl["net"]
    what = {2: "cfg2: 20-qubit QAOA cut network (3 subcircuits, K=5), full 2^20 distribution",
            3: "cfg3: 30-qubit ansatz cut network (3 subcircuits, K=6)",
            4: "cfg4: 64-qubit 8x8-grid cut network (8 subcircuits of 8 output qubits, K=14)",
            5: "cfg5: 196-qubit 14x14-grid cut network (52 subcircuits, c_s in 5..8)"}[wl["cfg"]]
    s = f"{what}; n={net.n_qubits} m={net.m} K={net.K}; seeded U[0,1) fp32 tensors"
    if wl["mode"] == "states":
        s += f"; batch of {wl['B']} uniform bitstrings"
        if wl["B"] != wl["full_B"]:
            s += f" (prefix of {wl['B']} of {wl['full_B']} states, SURVEY 8d-5)"
    return s


# ---------------------------------------------------------------------------------------------
# the CPU oracle legs (the only code here that touches oracle/)
# ---------------------------------------------------------------------------------------------
def oracle_sample_rate(wl, seconds: float, rank: int = 0, threads: int = 0):
    """Times the oracle AS IT STANDS on a bounded sample of the workload's states: the float64 direct sum over all
    4^K cut assignments (oracle/direct_sum.c, OpenMP over states) while 4^K is feasible, else the float64 per-state
    tensordot contraction O8' (oracle/reconstruct.py, numpy).  Returns (states/s, cores, sample description)."""
    from oracle import reconstruct as R
    from oracle.direct_sum_c import direct_sum_c
    net = wl["net"]
    cores = os.cpu_count() or 1
    if wl["mode"] == "states":
        bits_all = workload_states(wl, rank)
    else:
        idx = np.random.default_rng(1).choice(1 << net.n_qubits, size=min(1 << net.n_qubits, 1 << 16), replace=False)
        bits_all = ((idx[:, None] >> (net.n_qubits - 1 - np.arange(net.n_qubits))[None, :]) & 1).astype(np.uint8)
    T = wl["tensors"]
    if net.K <= 16:
        probe = min(len(bits_all), max(cores if threads == 0 else threads, 8 if threads == 0 else 1))
        t0 = time.perf_counter()
        _, used = direct_sum_c(net, T, bits_all[:probe], num_threads=threads)
        dt = max(time.perf_counter() - t0, 1e-6)
        n = int(min(len(bits_all), max(probe, probe * seconds / dt)))
        t0 = time.perf_counter()
        _, used = direct_sum_c(net, T, bits_all[:n], num_threads=threads)
        dt = time.perf_counter() - t0
        return n / dt, used, f"direct sum over 4^{net.K} cut assignments (C, OpenMP), first {n} states of the batch, {dt:.1f} s"
    # 4^K infeasible (cfg5, K = 152): the oracle's large-K tier O8' as it stands, per-state pairwise np.tensordot along
    # the oracle's own elimination order, numpy float64 (BLAS threads = host cores)
    order = R._elimination_order(net, trials=16)
    n, t0 = 0, time.perf_counter()
    while n < len(bits_all) and (n == 0 or time.perf_counter() - t0 < seconds):
        R.contract_states_tensordot(net, T, bits_all[n:n + 1], order=order)
        n += 1
    dt = time.perf_counter() - t0
    return n / dt, cores, (f"O8' per-state tensordot contraction (numpy float64; 4^K infeasible at K={net.K}), first {n} state(s) of "
                           f"the batch, {dt:.1f} s; cores = host threads available to BLAS")


def single_core_rate(wl, seconds: float):
    """The same oracle leg limited to one thread (BASELINE.md section 3 asks for both figures); None if it cannot be limited."""
    try:
        from threadpoolctl import threadpool_limits
    except ImportError:
        return None
    with threadpool_limits(limits=1):                      # numpy's BLAS; the C direct sum takes num_threads = 1
        rate, _cores, sample = oracle_sample_rate(wl, seconds, threads=1)
    return {"value": rate, "unit": UNIT, "cores": 1, "sample": sample}


def cpu_baseline(wl, seconds: float) -> dict:
    rate, cores, sample = oracle_sample_rate(wl, seconds)
    return {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
            "single_core": single_core_rate(wl, max(3.0, seconds / 3.0))}


def oracle_run(wl, bits, order=None):
    """One timed run of the oracle as it stands on the given states; returns (seconds, threads used)."""
    from oracle import reconstruct as R
    from oracle.direct_sum_c import direct_sum_c
    t0 = time.perf_counter()
    if wl["net"].K <= 16:
        _, used = direct_sum_c(wl["net"], wl["tensors"], bits)
    else:
        R.contract_states_tensordot(wl["net"], wl["tensors"], bits, order=order)
        used = os.cpu_count() or 1
    return time.perf_counter() - t0, used


def run_reference(args) -> None:
    """The reference arm: the CPU oracle, as it stands, on rank 0's host cores; a step = a bounded sample of the batch."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import reconstruct as R
    wl = make_workload(args.workload, args.batch)
    net = wl["net"]
    cores = os.cpu_count() or 1
    if wl["mode"] == "states":
        bits_all = workload_states(wl, 0)
    else:
        idx = np.random.default_rng(1).choice(1 << net.n_qubits, size=min(1 << net.n_qubits, 1 << 16), replace=False)
        bits_all = ((idx[:, None] >> (net.n_qubits - 1 - np.arange(net.n_qubits))[None, :]) & 1).astype(np.uint8)
    order = R._elimination_order(net, trials=16) if net.K > 16 else None
    per_step = max(0.5, min(20.0, 150.0 / max(1, args.steps + args.warmup)))     # seconds of oracle work per step
    probe = 1 if net.K > 16 else min(len(bits_all), max(cores, 8))
    dt, used = oracle_run(wl, bits_all[:probe], order)
    n = int(max(probe, min(len(bits_all), probe * per_step / max(dt, 1e-6))))
    total, done = 0.0, 0
    for i in range(args.warmup + args.steps):
        lo = (i * n) % max(1, len(bits_all) - n + 1)
        dt, used = oracle_run(wl, bits_all[lo:lo + n], order)
        if i >= args.warmup:
            total += dt
            done += n
    value = done / total
    kind = ("direct sum over 4^%d cut assignments (C, OpenMP)" % net.K) if net.K <= 16 else \
           ("O8' per-state tensordot contraction (numpy float64; 4^K infeasible at K=%d)" % net.K)
    sample = f"{kind}; {args.steps} timed steps of {n} states each from the seeded batch, {total:.1f} s"
    n_out = wl["B"] if wl["mode"] == "states" else (1 << net.n_qubits)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
            "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_description(wl, None), "states_per_step_per_gpu": n,
                       "note": "CPU oracle on rank 0 only; a step is a bounded sample of the batch (states_per_step_per_gpu states)"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5", choices=["cfg2", "cfg3", "cfg4", "cfg5", "variants"],
                    help="variants: only the subcircuit-variant simulation row (secondary line, for profiling)")
    ap.add_argument("--batch", type=int, default=0, help="states per step per GPU (0: the config's own batch; for cfg5 "
                    "the SURVEY 8d-5 prefix: the smallest power of two whose step runs >= 1 s; 1000000 = the full cfg5 batch)")
    ap.add_argument("--restarts", type=int, default=-1, help="planner restarts with the run-time objective (0: deterministic "
                    "greedy; default: 1024 for cfg5, 0 otherwise)")
    ap.add_argument("--plan-seed", type=int, default=1)
    ap.add_argument("--table-log2", type=int, default=-1, help="cap on log2(entries) of a once-per-key table node (0: the library default, 24; "
                    "default: 30 for cfg5 - 4 GB tables, built once per call - and the library default otherwise)")
    ap.add_argument("--max-workspace-gb", type=int, default=64)
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-others", dest="others", action="store_false", help="skip the secondary workloads")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
