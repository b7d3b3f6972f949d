#!/usr/bin/env python
"""bench.py -- throughput of the CoS / SB-CoS hot path on B200 (contract: see DESIGN.md section 7).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--impl ours|reference]

One "step" = one pass of the whole hot path over one batch of synthetic configurations:
propagator tabulation (A2) -> layer propagation (A3) -> terminal readouts (A4); the DAG compile (A1)
happens once, outside the timed region.  `value` = configurations / s with the inputs (vertex sites and
times) resident in HBM; `e2e` = the same through cos_eval_host with HOST buffers (copies inside the timed
region).  N > 1 (torchrun): configurations are independent, so every rank runs its own batch (seed + rank),
no data-path collective ("weak" scaling, the default); `--scaling strong` cuts ONE global batch into per-rank slices
(paper_2507_12349_b200.sharding.shard_vertices) instead.  value = all ranks' configurations / max-over-ranks time.

`--impl reference` times the CPU oracle (oracle/) on the host cores on a bounded sample of the same
workload -- the paper ships no code, so the oracle is the reference arm.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from cos_workloads import draw_vertices, get_config  # noqa: E402
from cos_workloads.tables import table_for  # noqa: E402

METRIC = "connected_sum_configs_per_s"
UNIT = "configs/s"
# DRAM bytes (read + write) of the layer-kernel launches of ONE step from a committed `ncu --set full` capture of the
# SHIPPED kernels, per workload and batch: (bytes, batch, launches captured, source).  The value is a citation of that
# capture, not something this run measures; other workloads / batches report null.  Re-capture after any kernel change.
NCU_DRAM_BYTES_PER_STEP = {
    ("cfg4_square_sb3_n10", 8192): (244.663e9, 20, "profiles/r02b_layer_kernel_all_layers.md (ncu --set full, all 20 "
                                    "layer launches of one step, round-2 row kernel)"),
    ("cfg3_honeycomb_sb2_n10", 576): (377.628e9, 20, "profiles/r02b_layer_kernel_all_layers.md (ncu --set full, the 20 "
                                      "layer launches of one 576-configuration workspace chunk)"),
}
DEFAULT_WORKLOAD = "cfg4"       # n = 10: the order BASELINE.json's target is quoted on


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, help="cfg1..cfg5 (BASELINE.json configs, 1-based)")
    ap.add_argument("--batch", type=int, default=0, help="override the configuration count (0 = BASELINE's)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-alg3-baseline", action="store_true",
                    help="skip cpu_baseline_alg3 (literal Algorithm 3 in fp64 on the host, ~80 s at cfg4)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank its own full batch (default, the driver's run); strong = ONE global batch "
                         "cut into per-rank slices with sharding.shard_vertices")
    ap.add_argument("--no-other-workloads", action="store_true",
                    help="skip the short timings of the other BASELINE configurations (other_workloads block)")
    ap.add_argument("--layers", action="store_true", help="print the per-layer table to stderr")
    ap.add_argument("--tune", action="append", default=[], metavar="KEY=VALUE",
                    help="launch tuning through cos_set_tuning (prefetch, warps_per_cta, blocks_per_cta_cap, pdl, ...)")
    ap.add_argument("--route", default="dag", choices=["dag", "det"],
                    help="dag: the hot path (default, the driver's contract); det: the determinant-polynomial route "
                         "cos_det_eval (SURVEY 8(f).3) on the same workload, all 2^n-1 subsets, its own JSON line")
    ap.add_argument("--precision", default="dd", choices=["fp64", "dd"], help="--route det: working precision")
    ap.add_argument("--order", type=int, default=0, help="--route det: override the order n (0 = the workload's)")
    return ap.parse_args()


def workload_of(args, rank=0):
    w = get_config(int(args.workload.replace("cfg", "")))
    kw = {"seed": w.seed + 1000 * rank}
    if args.batch:
        kw["batch"] = args.batch
    return w.scaled(**kw)


def config_dict(w, n_gpus, extra=None, global_batch=None):
    """global_batch: the one batch that was cut over the ranks (--scaling strong); None = every rank ran w.batch."""
    c = {"workload": w.name, "n": w.n, "n_flavors": w.n_flavors, "lattice": "honeycomb" if w.lattice else "square",
         "mode": "uniform" if w.alphas is None else "sb", "all_subsets": w.all_subsets, "batch_per_gpu": w.batch,
         "global_batch": w.batch * n_gpus if global_batch is None else global_batch,
         "L": w.L, "beta": w.beta, "n_tau": w.n_tau, "seed": w.seed,
         "parallelism": ("independent batches x%d (one per rank, seed + 1000 rank), no collective" % n_gpus)
                        if global_batch is None else
                        ("one global batch cut into %d contiguous slices (shard_vertices), no collective" % n_gpus)}
    if extra:
        c.update(extra)
    return c


# ------------------------------------------------------------------------------------------ CPU oracle timing
def _oracle_one(task):
    """One configuration through the cheapest oracle tier that returns the workload's outputs."""
    import oracle
    G, n, n_sub, nf, sigmas, uniform, all_subsets = task
    if uniform and n_sub == 1:
        return oracle.o3_uniform(G[0], nf, 0.0, all_subsets)          # printed recurrence Eq. 8-15
    if not uniform and n_sub == 1 and not all_subsets:
        return oracle.o2b_polynomial(G, sigmas)[-1:]                  # polynomial route Eq. 34-38
    tier = "o2a" if nf == 2 else "o2b"
    return oracle.connected_reference(G, n, n_sub, nf, sigmas, uniform, all_subsets, tier=tier)


def oracle_tier_name(w):
    """The cheapest oracle tier that returns the workload's outputs.  BASELINE.md section 3 names the fp64 O3 recurrences
    as the CPU evaluator; for the SB workloads at n = 10 literal Algorithm 3 costs ~78 s per configuration and core (cfg4;
    2^10 sublattice assignments times that for cfg3), outside the bounded-sample budget, so the determinant routes
    (binary128 arithmetic, 14-16 s per configuration and core) are timed there -- they are the FASTER CPU program."""
    if w.alphas is None and w.n_sub == 1:
        return "O3 uniform rooted recurrence (Eq. 8-15), fp64"
    if w.alphas is not None and w.n_sub == 1 and not w.all_subsets:
        return "O2b determinant-polynomial route (Eq. 34-38), binary128 (cheaper than O3 / Algorithm 3 fp64 at this size)"
    return "sum over sublattice assignments of %s, binary128" % ("O2a' two-determinant CDet" if w.n_flavors == 2 else "O2b")


def time_oracle(w, n_sample, procs):
    """Times the oracle as it stands on `n_sample` configurations of workload `w`, `procs` processes.
    Returns (configs/s, seconds)."""
    import multiprocessing as mp
    import oracle
    oracle.build_oracle()
    ws = w.scaled(batch=n_sample)
    table = table_for(ws)
    v = draw_vertices(ws)
    G = oracle.tabulate_reference(table, v["sites"], v["tau"])
    tasks = [(np.ascontiguousarray(G[..., c]), w.n, w.n_sub, w.n_flavors, w.sigmas, w.alphas is None, w.all_subsets)
             for c in range(n_sample)]
    t0 = time.perf_counter()
    if procs > 1:
        with mp.get_context("fork").Pool(procs) as pool:
            pool.map(_oracle_one, tasks, chunksize=1)
    else:
        for t in tasks:
            _oracle_one(t)
    dt = time.perf_counter() - t0
    return n_sample / dt, dt


def _alg3_one(task):
    import oracle
    G, sigmas = task
    return oracle.o3_alg3(G, sigmas)


def time_alg3(w, procs):
    """The paper's own recurrence on the host ("the practical CPU evaluator"): literal Algorithm 3
     in fp64, oracle.o3_alg3 as it stands, ONE configuration of workload `w` per process.
    Returns (configs/s, seconds)."""
    import multiprocessing as mp
    import oracle
    oracle.build_oracle()
    ws = w.scaled(batch=procs)
    table = table_for(ws)
    v = draw_vertices(ws)
    G = oracle.tabulate_reference(table, v["sites"], v["tau"])
    tasks = [(np.ascontiguousarray(G[..., c]), w.sigmas) for c in range(procs)]
    t0 = time.perf_counter()
    with mp.get_context("fork").Pool(procs) as pool:
        pool.map(_alg3_one, tasks, chunksize=1)
    dt = time.perf_counter() - t0
    return procs / dt, dt


ORACLE_SECONDS_PER_CONFIG = {"cfg1": 2e-4, "cfg2": 0.12, "cfg3": 16.0, "cfg4": 12.0, "cfg5": 16.0}   # rough, one core


def oracle_sample_plan(args, target_core_seconds=20.0):
    cores = os.cpu_count() or 1
    procs = max(1, min(cores, 16))
    per = ORACLE_SECONDS_PER_CONFIG.get(args.workload, 1.0)
    n = int(max(procs, min(4096, target_core_seconds * procs / per / 4)))
    n = max(procs, (n // procs) * procs)
    if per * n / procs > 60:
        n = procs
    return n, procs


# ------------------------------------------------------------------------------------------ clocks sampling
class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------ reference arm
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = workload_of(args)
    n_sample, procs = oracle_sample_plan(args, target_core_seconds=8.0)
    rates = []
    for _ in range(args.warmup):
        time_oracle(w, procs, procs)
    t_total = 0.0
    for _ in range(args.steps):
        r, dt = time_oracle(w, n_sample, procs)
        rates.append(r); t_total += dt
    value = n_sample * args.steps / t_total
    sample = "%d configurations of %s per step, %s, %d processes" % (n_sample, w.name, oracle_tier_name(w), procs)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(w, 1, {"sample_per_step": n_sample}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": procs, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------ our arm
def quick_measure(cos, torch, cfg, steps, warmup, peak_gbs, local_rank):
    """Short device-resident timing of another BASELINE configuration at its full size (same step: tabulate + evaluate):
    ms per step, configurations/s, whole-step fraction of the HBM roofline, clocks."""
    w = get_config(cfg)
    table = table_for(w)
    v = draw_vertices(w)
    tab = cos.cos_tab_build(w.lattice, w.L, table.n_blocks, w.beta, w.n_tau, table.data)
    h = cos.cos_build(w.n, w.n_flavors, w.lattice, w.sigmas, w.n if w.all_subsets else 0)
    try:
        info = cos.dag_summary(h)
        B = w.batch
        n_slots = info["n_blocks"] * info["d"] ** 2
        dev = torch.device("cuda", local_rank)
        sites, tau = torch.from_numpy(v["sites"]).to(dev), torch.from_numpy(v["tau"]).to(dev)
        G = torch.empty((n_slots, B), dtype=torch.float64, device=dev)
        out = torch.empty((w.n_out, B), dtype=torch.float64, device=dev)
        stream = torch.cuda.current_stream()
        cos.cos_reserve(h, B)
        for _ in range(warmup):
            cos.cos_tabulate(tab, w.n, sites, tau, B, G, stream)
            cos.cos_eval(h, G, B, out, stream)
        torch.cuda.synchronize()
        sampler = ClockSampler(local_rank)
        sampler.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            cos.cos_tabulate(tab, w.n, sites, tau, B, G, stream)
            cos.cos_eval(h, G, B, out, stream)
        e1.record(stream)
        torch.cuda.synchronize()
        clocks = sampler.stop()
        ms = e0.elapsed_time(e1) / steps
        assert bool(torch.isfinite(out).all())
        alg = (16 * info["n_states"] + 8 * n_slots + 8 * w.n_out) * B + info["program_bytes"]
        return {"workload": w.name, "n": w.n, "batch": B, "steps": steps, "warmup": warmup, "ms_per_step": ms,
                "configs_per_s": B / (ms * 1e-3),
                "edge_evals_per_s": (info["n_edges"] + info["n_readout_edges"]) * B / (ms * 1e-3),
                "algorithmic_bytes_per_step": alg, "frac_whole_step": alg / (ms * 1e-3) / (peak_gbs * 1e9),
                "clocks": clocks}
    finally:
        cos.cos_free(h)
        cos.cos_tab_free(tab)


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2507_12349_b200 as cos

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    use_dist = world > 1 or bool(os.environ.get("COS_BENCH_FORCE_DIST"))     # the latter: exercise NCCL with one rank
    json_out = sys.stdout
    if use_dist:
        # stdout carries the one JSON line and nothing else: NCCL prints its version banner to file descriptor 1 when the
        # communicator is created, so fd 1 points at stderr from here on and the line goes to a duplicate of the real one
        sys.stdout.flush()
        json_out = os.fdopen(os.dup(1), "w")
        os.dup2(2, 1)
        dist.init_process_group("nccl", device_id=dev)
    cos.load_library()

    strong = args.scaling == "strong"
    if strong:
        # one global batch, the same on every rank (same seed); this rank evaluates its contiguous slice only
        from paper_2507_12349_b200.sharding import shard_vertices
        w_global = workload_of(args, 0)
        global_B = w_global.batch
        _, _, v = shard_vertices(draw_vertices(w_global), global_B, rank, world)
        w = w_global.scaled(batch=v["tau"].shape[-1])
        if w.batch == 0:
            raise SystemExit("--scaling strong: the global batch has fewer configurations than ranks")
    else:
        w = workload_of(args, rank)
        global_B = None
        v = draw_vertices(w)
    B = w.batch
    total_B = global_B if strong else world * B          # configurations all ranks process per step
    table = table_for(w)
    tab = cos.cos_tab_build(w.lattice, w.L, table.n_blocks, w.beta, w.n_tau, table.data)
    t0 = time.perf_counter()
    h = cos.cos_build(w.n, w.n_flavors, w.lattice, w.sigmas, w.n if w.all_subsets else 0)
    build_s = time.perf_counter() - t0
    for kv in args.tune:
        k, val = kv.split("=")
        cos.cos_set_tuning(h, k, int(val))
    info = cos.dag_summary(h)
    NL = info["n_layers"]
    n_slots = info["n_blocks"] * info["d"] ** 2

    sites_h = torch.from_numpy(v["sites"]).pin_memory()
    tau_h = torch.from_numpy(v["tau"]).pin_memory()
    out_h = torch.empty((w.n_out, B), dtype=torch.float64).pin_memory()
    sites = sites_h.to(dev)
    tau = tau_h.to(dev)
    G = torch.empty((n_slots, B), dtype=torch.float64, device=dev)
    out = torch.empty((w.n_out, B), dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream()

    def step():
        cos.cos_tabulate(tab, w.n, sites, tau, B, G, stream)
        cos.cos_eval(h, G, B, out, stream)

    def barrier():
        torch.cuda.synchronize()
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    cos.cos_reserve(h, B)               # cos_eval then only enqueues kernels
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()

    # ---- timed region 1: device-resident inputs, the launch configuration a user gets (no per-layer events)
    launches0 = cos.cos_info(h, "n_launches")
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    launches = cos.cos_info(h, "n_launches") - launches0 + args.steps      # + one tabulation launch per step

    # ---- timed region 1b: the same steps with CUDA events recorded around every layer launch inside cos_eval (on its
    # stream): duration of the dominant kernel for the roofline.  Per-layer events serialise the layers (no PDL overlap).
    cos.cos_set_profiling(h, True)
    cos.cos_get_layer_times(h)                      # clear
    ev4, ev5 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev4.record(stream)
    for _ in range(args.steps):
        step()
    ev5.record(stream)
    barrier()
    ms_profiled = ev4.elapsed_time(ev5)
    clocks = sampler.stop() if rank == 0 else None
    layer_ms, n_prof = cos.cos_get_layer_times(h)
    cos.cos_set_profiling(h, False)

    # ---- timed region 2: end to end through the C-ABI with host buffers
    for _ in range(2):
        cos.cos_eval_host(h, tab, sites_h, tau_h, B, out_h, stream)
    barrier()
    ev2, ev3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev2.record(stream)
    for _ in range(args.steps):
        cos.cos_eval_host(h, tab, sites_h, tau_h, B, out_h, stream)
    ev3.record(stream)
    barrier()
    ms_e2e = ev2.elapsed_time(ev3)
    assert torch.equal(out_h, out.cpu()), "host-buffer pipeline and device pipeline disagree"
    assert bool(torch.isfinite(out_h).all())

    from paper_2507_12349_b200.sharding import max_over_ranks
    ms_total, ms_e2e, layer_sum = max_over_ranks([ms_total, ms_e2e, sum(layer_ms)], device=dev)

    if rank == 0:
        K = args.steps
        value = total_B * K / (ms_total * 1e-3)
        e2e_value = total_B * K / (ms_e2e * 1e-3)
        edges = info["n_edges"] + info["n_readout_edges"]
        # ---- roofline of the dominant kernel (cos_layer_kernel, NL launches per step); DESIGN.md section 6
        S = info["n_states"]
        alg_bytes_step = (16 * S + 8 * n_slots + 8 * w.n_out) * B + info["program_bytes"]
        # Duration of the dominant kernel per step: its SHARE of a step comes from the profiled pass (CUDA events around
        # every layer launch, which serialise the layers and cost a little), the step time from the unprofiled region
        # (CUDA events around the K timed steps on the launching stream): kernel time = step time x share.
        layer_s_profiled = layer_sum * 1e-3 / max(n_prof, 1)
        share = min(1.0, layer_s_profiled * 1e3 / (ms_profiled / K))
        layer_s_step = (ms_total / K) * 1e-3 * share
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
            peak_gbs, peak_src = float(peaks["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
        except (OSError, KeyError, ValueError):
            peak_gbs, peak_src = 6650.0, "fallback (B200_PROFILING.md)"
        achieved_gbs = alg_bytes_step / layer_s_step / 1e9
        traffic, traffic_src = None, None
        cap = NCU_DRAM_BYTES_PER_STEP.get((w.name, B))
        if cap:
            traffic, traffic_src = cap[0] / cap[1], cap[2] + "; per launch = captured total / %d launches" % cap[1]
        fma_peak = cos.cos_measure_fp64_fma_peak()
        t_hbm = alg_bytes_step / (peak_gbs * 1e9)
        t_fp64 = info["n_fma"] * B / fma_peak
        roofline = {"bound": "hbm" if t_hbm >= t_fp64 else "alu", "kernel": "cos_layer_kernel",
                    "achieved": achieved_gbs, "peak": peak_gbs, "unit": "GB/s", "frac": achieved_gbs / peak_gbs,
                    "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": alg_bytes_step / NL,
                    "launches_per_step": NL, "kernel_ms_per_step": layer_s_step * 1e3,
                    "kernel_share_of_step": share, "kernel_ms_per_step_profiled": layer_s_profiled * 1e3,
                    "profiled_ms_per_step": ms_profiled / K,
                    "frac_whole_step": t_hbm * 1e3 / (ms_total / K),   # roofline time / unprofiled step (all kernels)
                    "algorithmic_bytes_per_step": alg_bytes_step,
                    "t_roofline_hbm_ms": t_hbm * 1e3, "t_roofline_fp64_ms": t_fp64 * 1e3,
                    "fp64_fma_peak_measured_tflops": 2 * fma_peak / 1e12,
                    "fp64_fma_achieved_tflops": 2 * info["n_fma"] * B / layer_s_step / 1e12}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
                "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": config_dict(w, world, global_batch=global_B, extra={"l2": "inputs larger than L2: the two layer slabs hold %.1f GB per step"
                                                 % (16 * info["max_layer_states"] * B / 1e9),
                                                 "dag": {k: info[k] for k in ("n_states", "n_edges", "n_readout_edges",
                                                                               "n_fma", "max_layer_states", "program_bytes")},
                                                 "build_s": build_s}),
                "edge_evals_per_s": total_B * edges * K / (ms_total * 1e-3),
                "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": ms_e2e / K,
                        "h2d_bytes_per_step": B * w.n * (2 * 4 + 8), "d2h_bytes_per_step": B * w.n_out * 8},
                "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline}
        if world == 1 and not args.no_other_workloads and args.workload == DEFAULT_WORKLOAD and not args.batch:
            # the other n = 10 configuration (cfg3, the larger and weaker one) and cfg2 / cfg5 / cfg1, driver-timed in the
            # same run: short timings (>= 3 warm-up steps), whole-step roofline fraction; not the headline `value`
            # (the headline handle's workspace is released first: cfg3 needs the default 64 GiB workspace of its own; a
            # workload that fails, e.g. for lack of free device memory, is reported as such and never costs the line)
            cos.cos_free(h)
            h = None
            del G, out
            torch.cuda.empty_cache()
            others = []
            for c, k in ((3, 3), (2, 10), (5, 20), (1, 50)):
                try:
                    others.append(quick_measure(cos, torch, c, k, 3, peak_gbs, local_rank))
                except Exception as exc:       # noqa: BLE001 -- report, do not lose the headline line
                    others.append({"workload": get_config(c).name, "error": str(exc)[:200]})
                    torch.cuda.empty_cache()
            line["other_workloads"] = others
        if not args.no_cpu_baseline and world == 1:
            n_sample, procs = oracle_sample_plan(args)
            rate, dt = time_oracle(workload_of(args), n_sample, procs)
            line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": procs, "kind": "oracle", "seconds": dt,
                                    "tier": oracle_tier_name(w),
                                    "sample": "%d configurations of %s, %s" % (n_sample, w.name, oracle_tier_name(w))}
            # the paper's own algorithm on the host cores as well (square-lattice SB workloads: ~80 s for one configuration
            # per core at n = 10; the honeycomb workload would need 2^10 times that per configuration and is left out)
            if w.alphas is not None and w.n_sub == 1 and not w.all_subsets and not args.no_alg3_baseline:
                rate3, dt3 = time_alg3(workload_of(args), procs)
                line["cpu_baseline_alg3"] = {"value": rate3, "unit": UNIT, "cores": procs, "kind": "oracle", "seconds": dt3,
                                             "tier": "O3 literal Algorithm 3 (PAPER.md:546-595), fp64",
                                             "sample": "%d configurations of %s, one per process" % (procs, w.name)}
        if args.layers:
            sys.stderr.write("layer  states      ms/step   GB/s(alg)\n")
            for l in range(NL):
                s_in = info["layer_states"][l]
                s_out = info["layer_states"][l + 1] if l + 1 < NL else 0
                ms = layer_ms[l] / max(n_prof, 1)
                gb = 8.0 * (s_in + s_out) * B / 1e9
                sys.stderr.write("%3d %10d %10.4f %10.1f\n" % (l, s_in, ms, gb / (ms * 1e-3) if ms > 0 else 0.0))
        json_out.write(json.dumps(line) + "\n")
        json_out.flush()

    if h is not None:
        cos.cos_free(h)
    cos.cos_tab_free(tab)
    if use_dist:
        dist.barrier()
        dist.destroy_process_group()


def run_det(args):
    """Secondary workload (not the driver's line): tabulate -> cos_det_eval on a square-lattice workload; one step =
    all 2^n-1 connected values of every configuration by Eq. 34-38.  ALU-bound: achieved = terms of Eq. 36 + Eq. 38 per
    second against the measured fp64 FMA peak (one fp64 FMA per term in fp64; a double-double multiply-add is ~25 fp64
    operations, so the dd fraction is reported against the same peak and is correspondingly small)."""
    import torch
    import paper_2507_12349_b200 as cos
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    cos.load_library()
    w = workload_of(args)
    if args.order:
        w = w.scaled(n=args.order)
    n, B, nf, nb = w.n, w.batch, w.n_flavors, w.n_blocks
    prec = cos.COS_DET_DD if args.precision == "dd" else cos.COS_DET_FP64
    table = table_for(w)
    v = draw_vertices(w)
    tab = cos.cos_tab_build(w.lattice, w.L, table.n_blocks, w.beta, w.n_tau, table.data)
    sites, tau = torch.from_numpy(v["sites"]).to(dev), torch.from_numpy(v["tau"]).to(dev)
    G = torch.empty((nb * w.d * w.d, B), dtype=torch.float64, device=dev)
    out = torch.empty(((1 << n) - 1, B), dtype=torch.float64, device=dev)
    work = torch.empty((cos.cos_det_workspace_bytes(n, nb, prec, B) + 7) // 8, dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream()

    def step():
        cos.cos_tabulate(tab, n, sites, tau, B, G, stream)
        cos.cos_det_eval(n, nf, nb, w.sigmas, prec, G, B, out, work, stream, lattice=w.lattice)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = ev0.elapsed_time(ev1) / args.steps
    assert bool(torch.isfinite(out).all())
    # terms of Eq. 36 with a non-vanishing weight: per site of T one of the N_f(N_f-1)/2 flavour pairs or one of the
    # flavours whose sigma is not zero (a zero sigma removes that choice from the loops) -> (1 + pairs + singles)^n - 1
    n_single = sum(1 for x in (w.sigmas or ()) if x != 0.0)
    terms36 = (1 + nf * (nf - 1) // 2 + n_single) ** n - 1
    sg = tuple(w.sigmas or (0.0,) * nf)
    if nf == 3 and sg[1] == 0.0:
        # sigma_1 = 0: the sums over d_1 and d_2 factorise (cos_det.cu): per (S_0, X) 2^|free F_0| + 2^|free U| terms
        o0, oy = (2 if sg[0] != 0.0 else 1), (2 if sg[2] != 0.0 else 1)
        terms36 = (3 + o0) ** n + (3 + oy) ** n - 2
    n_assign = 2 ** n if w.lattice == 1 else 1          # honeycomb: every sublattice assignment is walked
    terms36 *= n_assign
    terms38 = (3 ** n - 1) // 2 - (2 ** n - 1)
    fma_peak = cos.cos_measure_fp64_fma_peak()
    achieved = (terms36 + terms38) * B / (ms * 1e-3)
    line = {"metric": "det_route_configs_per_s", "value": B / (ms * 1e-3), "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64" if prec == 0 else "f64x2 (double-double)",
            "data": "synthetic",
            "config": config_dict(w, 1, {"route": "determinant-polynomial Eq. 34-38, all %d subsets" % ((1 << n) - 1),
                                         "terms_eq36_per_config": terms36, "terms_eq36_all_sigma_nonzero": (1 + nf * (nf + 1) // 2) ** n - 1, "terms_eq38_per_config": terms38,
                                         "workspace_bytes": work.numel() * 8,
                                         "l2": "minors + moments per step: %.2f GB" % (work.numel() * 8 / 1e9)}),
            "gpu_launches": (3 + 2 * n_assign) * args.steps, "clocks": clocks,
            "roofline": {"bound": "alu", "kernel": "cos_det_moment_kernel", "achieved": achieved / 1e9,
                         "peak": fma_peak / 1e9, "unit": "GFMA/s (terms of Eq. 36 + 38 vs fp64 FMA peak)",
                         "frac": achieved / fma_peak, "traffic": None,
                         "peak_source": "cos_measure_fp64_fma_peak (measured in this run)"}}
    print(json.dumps(line), flush=True)
    cos.cos_tab_free(tab)


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.route == "det":
        run_det(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
