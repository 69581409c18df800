"""bench.py -- cell-updates/s of the THOR HE-VI large step on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W]            the CUDA path (default N = 1)
  python bench.py --impl reference [--steps K] [--warmup W]      the oracle on the host cores

A "step" is one large time step (all rows of DESIGN.md's hot-path table: three Runge-Kutta stages
of slow terms + 1 + n/2 + n acoustic substeps + forcing) of config 3 of BASELINE.json
(level 6 x 32 layers, hot-Jupiter constants, n = 8): 40962 x 32 cells x 13 substeps per step.
One JSON line on stdout (rank 0).  Multi-GPU: the path is fixed to one GPU by north_star
("replicas only"): every rank runs an independent replica, no data-path collective.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import thor_inputs as ti  # noqa: E402

WORKLOAD = 3
METRIC = "cell-updates/s (cols x layers x acoustic substeps) FP64"
UNIT = "cell-updates/s"

# algorithmic bytes per cell per launch (DESIGN.md section 8 "byte budget"); geometry bytes are per column
K2_SURVEY_DOUBLES = 18   # k_vertical's share of SURVEY 8(d)'s 27 doubles: 14 reads (V*'(3) re-read, p*, W*, rho*,
                         # rho-theta, 4 slow terms, rho^t, p^t, theta^t) + 4 writes
K2_DESIGN_DOUBLES = 19   # what this design's kernel moves once per cell: 15 reads (V*' as 2 tangent components, h,
                         # theta, rho*, W*, (rho theta)*, 4 slow terms, 3 LU factors, p^t) + 4 writes
K1_SURVEY_DOUBLES = 10   # k_momentum's share: p*, V*(3), slowV(3) read; V*'(3) written
K1_DESIGN_DOUBLES = 7    # p*, V*(2), slowV(2) read; V*'(2) written
SUBSTEP_SURVEY_DOUBLES = 27   # B_dep of SURVEY 8(d) = the figure the 60 % target is stated on
SUBSTEP_DESIGN_DOUBLES = K1_DESIGN_DOUBLES + K2_DESIGN_DOUBLES
SURVEY_GEOM_BYTES = 336       # per column, SURVEY 8(d)
K2_GEOM_BYTES = 8 * 4 + 16 * 8    # this design: 8 int32 neighbour slots + 7x2 (+2 pad) contracted divergence weights
K1_GEOM_BYTES = 8 * 4 + 12 * 8    # 8 int32 + 6x2 contracted gradient weights
# HBM traffic per launch, WARM (ncu --cache-control none over graph-replayed large steps, so every kernel finds
# the L2 as its predecessor left it -- the situation bench.py times): raw ncu csv committed under profiles/,
# the command that wrote it in the .md beside it.  Parsed here, never typed in.
WARM_TRAFFIC_CSV = {3: "profiles/r02_warm_traffic_cfg3.csv", 4: "profiles/r02_warm_traffic_cfg4.csv"}


def ncu_warm_traffic(workload, kernel_prefix):
    """Mean dram__bytes_read.sum + dram__bytes_write.sum per launch of the kernels whose name starts with
    `kernel_prefix` in the committed raw ncu csv of `workload` (None if there is no such file or kernel)."""
    import csv
    path = os.path.join(ROOT, WARM_TRAFFIC_CSV.get(workload, ""))
    if not os.path.isfile(path):
        return None
    per_launch = {}
    with open(path, newline="") as f:
        rows = [r for r in f if r.startswith('"')]
    rd = csv.reader(rows)
    head = next(rd, None)
    if not head or "Metric Name" not in head:
        return None
    i_id, i_k, i_m, i_v = head.index("ID"), head.index("Kernel Name"), head.index("Metric Name"), head.index("Metric Value")
    for r in rd:
        name = r[i_k]
        for pre in ("void ", "thor::"):
            if name.startswith(pre):
                name = name[len(pre):]
        if name.startswith(kernel_prefix + "<") or name.startswith(kernel_prefix + "("):
            if r[i_m] in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                per_launch[r[i_id]] = per_launch.get(r[i_id], 0.0) + float(r[i_v].replace(",", ""))
    return sum(per_launch.values()) / len(per_launch) if per_launch else None


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.stop_flag = index, [], threading.Event()

    def run(self):
        while not self.stop_flag.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                parts = [x.strip() for x in out.strip().split(",")]
                if len(parts) >= 7:
                    self.samples.append(parts)
            except Exception:
                pass
            self.stop_flag.wait(0.1)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(s[0]) for s in self.samples)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(s[3 + i].lower().startswith("active") for s in self.samples)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.samples[0][1]), "reasons": reasons,
                "samples": len(sm), "power_w_max": max(float(s[2]) for s in self.samples)}


def max_over_ranks(values, device="cpu"):
    """Element-wise MAX of a list of floats over all ranks (the timing rule for N > 1).  Works with
    any initialised torch.distributed backend (nccl on the GPU box, gloo in the CPU tests); without
    a process group it is the identity."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor(list(values), device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def aggregate_value(cells_per_step, steps, world, ms):
    """Whole-job throughput of `world` independent replicas (weak scaling, no data-path collective):
    units all ranks processed / the slowest rank's time."""
    return cells_per_step * steps * world / (ms * 1e-3)


def oracle_sample_level(workload):
    """Grid level of the oracle-timing legs: the workload's own up to level 6 (0.45 s per large step on 16
    cores at config 3); config 4's level 7 x 64 costs ~5 s per step, so it is sampled at level 6 with dt doubled."""
    return min(ti.CONFIGS[workload]["level"], 6)


def time_oracle(workload, n_steps, warmup, threads=None):
    """The oracle as it stands on the host cores -- nothing of the product is imported, loaded or called here.
    The grid is the oracle's own generator WITHOUT spring smoothing (level 6 smoothing in numpy would take
    minutes; the oracle's work per step does not depend on where the points sit).  threads=None: all cores."""
    import oracle
    from oracle import grid_oracle
    cfg = dict(ti.CONFIGS[workload])
    level = oracle_sample_level(workload)
    dt = cfg["dt"] * 2 ** (cfg["level"] - level)
    xyz, nbr, C, _ = grid_oracle.build(level, smooth=False)
    G = oracle.Geometry(xyz, nbr, cfg["nv"], cfg["planet"], C)
    state = ti.initial_state(workload, xyz)
    F = ti.forcing_tables(workload, xyz)
    all_threads = oracle.num_threads()
    if threads is not None:
        oracle.set_num_threads(threads)
    try:
        for _ in range(warmup):
            state = G.step(*state, 1, dt, cfg["n_sub"], F)
        t0 = time.perf_counter()
        for _ in range(n_steps):
            state = G.step(*state, 1, dt, cfg["n_sub"], F)
        el = time.perf_counter() - t0
        used = oracle.num_threads()
    finally:
        oracle.set_num_threads(all_threads)
    cells = xyz.shape[0] * cfg["nv"] * ti.substeps_per_large_step(cfg["n_sub"])
    sample = "config %d at level %d x %d layers (%d columns, unsmoothed bisection grid of the oracle's own generator), " \
             "%d large steps of dt=%g s, n=%d, forcing tables on" % (workload, level, cfg["nv"], xyz.shape[0], n_steps, dt, cfg["n_sub"])
    return cells * n_steps / el, el / max(n_steps, 1), used, sample


def time_oracle_operators(workload, reps=3):
    """Config 1's stencils (Eq. 6, Eq. 7) as the oracle evaluates them, timed alone on the host cores on the
    grid size of `workload`: seconds per application, all cores; oracle/ only."""
    import oracle
    from oracle import grid_oracle
    cfg = ti.CONFIGS[workload]
    level = oracle_sample_level(workload)
    xyz, nbr, C, _ = grid_oracle.build(level, smooth=False)
    G = oracle.Geometry(xyz, nbr, cfg["nv"], cfg["planet"], C)
    rng = np.random.default_rng(ti.SEED0)
    s = rng.standard_normal((xyz.shape[0], cfg["nv"]))
    v = rng.standard_normal((xyz.shape[0], cfg["nv"], 3))
    out = {}
    for name, fn, arg in (("div", G.hdiv, v), ("grad", G.hgrad, s), ("lap", G.hlap, s)):
        fn(arg)
        t0 = time.perf_counter()
        for _ in range(reps):
            fn(arg)
        out[name] = (time.perf_counter() - t0) / reps
    return out, oracle.num_threads(), level


def workload_config(workload, N, world):
    """The `config` object both arms print (same workload, same words)."""
    cfg = ti.CONFIGS[workload]
    nv, n = cfg["nv"], cfg["n_sub"]
    substeps = ti.substeps_per_large_step(n)
    cells = N * nv
    return {"workload": "config %d: level %d (%d columns) x %d layers, hot-Jupiter constants, dt=%g s, "
                        "n=%d (%d substeps per large step), Newtonian relaxation forcing" % (
                            workload, cfg["level"], N, nv, cfg["dt"], n, substeps),
            "cells": cells, "substeps_per_step": substeps, "parallelism": "replicas x%d" % world}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    value, per_step, cores, sample = time_oracle(WORKLOAD, args.steps, args.warmup)
    v1, _, _, _ = time_oracle(WORKLOAD, 1, 0, threads=1)
    level = oracle_sample_level(WORKLOAD)
    config = workload_config(WORKLOAD, ti.n_columns(level), 1)
    if level != ti.CONFIGS[WORKLOAD]["level"]:
        config["workload"] += " -- SAMPLED by the oracle arm: " + sample
    config["oracle_grid"] = "unsmoothed bisection grid of the oracle's own generator (no product code in this arm)"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": per_step * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "value_1_thread": v1},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_cuda(args):
    import torch
    import torch.distributed as dist
    import paper_1607_05535_b200 as thor

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback (use --impl reference)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = ti.CONFIGS[WORKLOAD]
    nv, dt, n = cfg["nv"], cfg["dt"], cfg["n_sub"]
    grid = thor.Grid(cfg["level"], nv, cfg["planet"])
    N = grid.n_cols
    xyz = grid.view["xyz"]
    host = ti.initial_state(WORKLOAD, xyz)
    forcing = ti.forcing_tables(WORKLOAD, xyz)
    stream = torch.cuda.Stream()
    state = thor.State(grid, *host, cuda_stream=stream.cuda_stream)
    substeps = ti.substeps_per_large_step(n)
    cells_per_step = N * nv * substeps

    if args.next1:
        state.set_diffusion(0.01992)
    with torch.cuda.stream(stream):
        for _ in range(max(args.warmup, 3)):
            state.step(1, dt, n, forcing)
        barrier()
        sampler = ClockSampler(local_rank)
        sampler.start()
        time.sleep(0.3)
        l0 = thor.thor_launch_count()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        ev0.record(stream)
        for _ in range(args.steps):
            state.step(1, dt, n, forcing)
        ev1.record(stream)
        barrier()
        launches = thor.thor_launch_count() - l0
        ms = ev0.elapsed_time(ev1)
        if args.step_only:                       # the profiling entry: nothing but large steps after set-up
            sampler.stop_flag.set()
            sampler.join()
            if rank == 0:
                print(json.dumps({"metric": METRIC, "value": aggregate_value(cells_per_step, args.steps, 1, ms), "unit": UNIT,
                                  "ms_per_step": ms / args.steps, "steps": args.steps, "gpu_launches": int(launches),
                                  "config": dict(workload_config(WORKLOAD, N, world), next1=bool(args.next1)),
                                  "note": "--step-only: the timed large steps alone (profiling entry), not a bench line"}), flush=True)
            if world > 1:
                dist.destroy_process_group()
            return

        # dominant kernel alone (K2 = divergences + column solve) and K1, CUDA events on the same stream.  Chunks of
        # n launches (a stage's worth) between untimed large steps, so that the timed state stays a physical one
        # (repeating one kernel alone for thousands of launches drives it to NaN and down another branch of
        # eos_dev); chunks are accumulated until the timed launches cover >= 0.2 s.
        def time_kernels(which, min_ms=200.0, chunk=n):
            state.step(1, dt, n, forcing)
            state.acoustic_substeps(chunk, dt / n, which)
            total, reps = 0.0, 0
            while total < min_ms and reps < 100000:
                state.step(1, dt, n, forcing)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                state.acoustic_substeps(chunk, dt / n, which)
                b.record(stream)
                b.synchronize()
                total += a.elapsed_time(b)
                reps += chunk
            return total / reps
        # config 1: the two stencils alone (Eq. 6, Eq. 7) on device arrays of this grid, 32 B/cell + geometry
        nc = N * nv
        bufs = [torch.rand(nc, dtype=torch.float64, device="cuda") for _ in range(7)]
        ptr = [b.data_ptr() for b in bufs]

        def time_op(fn, min_ms=200.0, chunk=200):
            for _ in range(3):
                fn()
            total, reps = 0.0, 0
            while total < min_ms:
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                for _ in range(chunk):
                    fn()
                b.record(stream)
                b.synchronize()
                total += a.elapsed_time(b)
                reps += chunk
            return total / reps
        div_ms = time_op(lambda: thor.thor_apply_div_device(grid.handle, ptr[0], ptr[1], ptr[2], ptr[3], stream.cuda_stream))
        grad_ms = time_op(lambda: thor.thor_apply_grad_device(grid.handle, ptr[0], ptr[4], ptr[5], ptr[6], stream.cuda_stream))
        lap_ms = time_op(lambda: thor.thor_apply_lap_device(grid.handle, ptr[0], ptr[3], stream.cuda_stream))
        del bufs
        k2_ms = time_kernels(2)
        k1_ms = time_kernels(1)
        sub_ms = time_kernels(3)
        sampler.stop_flag.set()
        sampler.join()

        # NEXT-1 switched on (hyper-diffusion + divergence damping, the paper's hot-Jupiter D): same step, extra kernels
        state.set(*host)
        state.set_diffusion(0.01992)
        for _ in range(3):
            state.step(1, dt, n, forcing)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record(stream)
        for _ in range(5):
            state.step(1, dt, n, forcing)
        b.record(stream)
        torch.cuda.synchronize()
        next1_ms = a.elapsed_time(b) / 5
        state.set_diffusion(0.0, 0.0)

        # end to end through the public API with host buffers: upload, step, download every step
        state.set(*host)
        pinned = [torch.from_numpy(a).pin_memory() for a in host]
        h_in = [t.numpy() for t in pinned]
        h_out = tuple(torch.empty_like(t).pin_memory().numpy() for t in pinned)
        state.set(*h_in)
        state.step(1, dt, n, forcing)
        state.get(h_out)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            state.set(*h_in)
            state.step(1, dt, n, forcing)
            state.get(h_out)
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - t0
        barrier()

    io_bytes = int(sum(a.nbytes for a in h_in))
    ms, e2e_s = max_over_ranks([ms, e2e_s], device="cuda")
    value = aggregate_value(cells_per_step, args.steps, world, ms)
    e2e_value = aggregate_value(cells_per_step, args.steps, world, e2e_s * 1e3)

    peak, peak_kind = measured_peak()
    cells = N * nv
    k2_bytes = cells * K2_SURVEY_DOUBLES * 8 + N * K2_GEOM_BYTES
    achieved = k2_bytes / (k2_ms * 1e-3) / 1e9
    sub_survey_bytes = cells * SUBSTEP_SURVEY_DOUBLES * 8 + N * SURVEY_GEOM_BYTES
    sub_design_bytes = cells * SUBSTEP_DESIGN_DOUBLES * 8 + N * (K1_GEOM_BYTES + K2_GEOM_BYTES)
    roofline = {"bound": "hbm", "kernel": "k_vertical (a5-a9: divergences + column solve + rho, rho-theta, p*)",
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": ncu_warm_traffic(WORKLOAD, "k_vertical"),
                "traffic_kind": "dram read + write bytes per launch, mean over the k_vertical launches of %s (ncu "
                                "--cache-control none over graph-replayed large steps: warm L2, as timed here)" % WARM_TRAFFIC_CSV.get(WORKLOAD),
                "bytes_model": "achieved/frac: k_vertical's share (18 doubles/cell) of SURVEY 8(d)'s 27-double budget; "
                               "achieved_design_bytes: the 19 doubles/cell this layout moves once",
                "peak_kind": peak_kind, "ms_per_launch": k2_ms, "bytes_per_launch": k2_bytes,
                "bytes_per_launch_design": cells * K2_DESIGN_DOUBLES * 8 + N * K2_GEOM_BYTES,
                "achieved_design_bytes": (cells * K2_DESIGN_DOUBLES * 8 + N * K2_GEOM_BYTES) / (k2_ms * 1e-3) / 1e9,
                "k1_ms_per_launch": k1_ms,
                "k1_achieved_survey_bytes": (cells * K1_SURVEY_DOUBLES * 8 + N * K1_GEOM_BYTES) / (k1_ms * 1e-3) / 1e9,
                "k1_achieved_design_bytes": (cells * K1_DESIGN_DOUBLES * 8 + N * K1_GEOM_BYTES) / (k1_ms * 1e-3) / 1e9,
                # the acoustic substep a4-a9 (both kernels back to back): what north_star's 60 % target is stated on
                "substep_ms": sub_ms,
                "substep_cell_updates_per_s": cells / (sub_ms * 1e-3),
                "substep_frac_survey_budget_of_measured_peak": sub_survey_bytes / (sub_ms * 1e-3) / 1e9 / peak,
                "substep_frac_survey_budget_of_8TBs": sub_survey_bytes / (sub_ms * 1e-3) / 1e9 / 8000.0,
                "substep_frac_design_bytes_of_measured_peak": sub_design_bytes / (sub_ms * 1e-3) / 1e9 / peak}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": dict(workload_config(WORKLOAD, N, world),
                           l2="one large step streams the 30-row column-record slab (%d MB) > 126 MB L2; no flush" % (
                               30 * 8 * cells * (64 if nv > 32 else 32) // nv // 1000000)),
            "clocks": sampler.summary(),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": io_bytes, "d2h_bytes_per_step": io_bytes,
                    "ms_per_step": e2e_s / args.steps * 1e3},
            "gpu_launches": int(launches), "roofline": roofline,
            "next1": {"what": "the same large step with NEXT-1 on (hyper-diffusion + 3-D divergence damping, D = 0.01992)",
                      "ms_per_step": next1_ms, "cell_updates_per_s": cells_per_step / (next1_ms * 1e-3)},
            "operators": {"what": "config 1 stencils alone on this grid (level %d x %d), device arrays, 32 B/cell + geometry" % (cfg["level"], nv),
                          "div_ms": div_ms, "div_GBs": (cells * 32 + N * 224) / (div_ms * 1e-3) / 1e9,
                          "grad_ms": grad_ms, "grad_GBs": (cells * 32 + N * 176) / (grad_ms * 1e-3) / 1e9,
                          "lap_ms": lap_ms, "lap_GBs": (cells * 16 + N * 96) / (lap_ms * 1e-3) / 1e9,
                          "lap_what": "horizontal Laplacian of L369-L371 (NEXT-1 building block), 16 B/cell + geometry"}}
    if world == 1 and not args.no_cpu_baseline:
        v, per, cores, sample = time_oracle(WORKLOAD, 4, 1)
        v1, _, _, _ = time_oracle(WORKLOAD, 1, 0, threads=1)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                                "value_1_thread": v1}
        ops, op_cores, op_level = time_oracle_operators(WORKLOAD)
        line["operators"].update({"oracle_div_ms": ops["div"] * 1e3, "oracle_grad_ms": ops["grad"] * 1e3,
                                  "oracle_lap_ms": ops["lap"] * 1e3, "oracle_cores": op_cores,
                                  "oracle_what": "the oracle's orc_hdiv / orc_hgrad / orc_hlap alone on level %d x %d "
                                                 "(unsmoothed grid of its own generator), all host cores" % (op_level, nv)})
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--step-only", action="store_true",
                    help="profiling entry: set up, warm up, run --steps large steps, print a short line and stop "
                         "(no kernel-alone loops, operators, NEXT-1 or e2e legs); the ncu commands under profiles/ use it")
    ap.add_argument("--next1", action="store_true", help="with --step-only: NEXT-1 on (D = 0.01992) in the timed steps")
    ap.add_argument("--workload", type=int, default=3, choices=[3, 4],
                    help="BASELINE.json config: 3 = level 6 x 32 (default, the configuration the target is stated on), "
                         "4 = level 7 x 64 (throughput at scale)")
    args = ap.parse_args()
    global WORKLOAD
    WORKLOAD = args.workload
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
