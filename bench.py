#!/usr/bin/env python
"""bench.py -- grid-point updates per second of the swept hot path on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path over one batch of synthetic input: one `swept_run` call that advances
the config-2 heat workload (FTCS, periodic, r = 0.25, 4 seeded sine modes; nx = 2^22, the largest nx of the sweep)
by `--nsteps` timesteps (default: the config's 50 000) -- remainder kernels, upright triangle, all diamonds and the
closing inverted triangle included.  value = nx * nsteps * K / (sum of the K CUDA-event step times).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--problem heat|ks|euler] [--dtype f64|f32] [--nx NX] [--nsteps NS] [--tile-width W] [--kernel wave|smem]
                    [--sweep]      (also time swept vs classic over nx = 2^11..2^22, written to gpurun_out/sweep_*.json)

N > 1 (torchrun, one rank per GPU): the path does not shard (north_star: one GPU, no collectives) -- every rank runs an
independent replica ("replicas only", scaling "weak"); value = units all ranks processed / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import workloads as wl  # noqa: E402

FP_INSTR_PER_STAGE_UPDATE = {  # thread-level FP-pipe instructions of one point update (DESIGN.md section 5.3 / 5.6)
    ("heat", "f64"): 3, ("heat", "f32"): 3, ("ks", "f64"): 11, ("ks", "f32"): 11,
    # Euler: SASS count of Euler<T>::group_sel (4 cells: 7 differences, 6 limited slopes, 5 face fluxes with IEEE
    # division and square root expanded inline) / 4: f64 (109 DADD + 199 DFMA + 145 DMUL + 44 DSETP) / 4,
    # f32 (122 FADD + 129 FFMA + 131 FMUL + 40 FSETP + 5 FMNMX) / 4
    ("euler", "f64"): 124.25, ("euler", "f32"): 106.75,
}


def kernel_sources_hash() -> str:
    """sha256 (first 16 hex digits) over the CUDA sources of the library: ties a stored ncu figure to the kernels it was taken from."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1612_02495_b200", "csrc")
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh", ".h")) and name not in ("heat2d.cu", "alu_peak.cu"):      # the 1-D path's sources
            h.update(name.encode())
            h.update(open(os.path.join(d, name), "rb").read())
    return h.hexdigest()[:16]


def traffic_of(args, w, W, chain):
    """(dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel's launch, where it comes from): read from the
    committed `ncu --set full` capture of this very configuration (profiles/traffic.csv names the report and the hash of the
    kernel sources it was captured from).  (None, why) if there is no capture, or if the kernel sources changed since."""
    try:
        import csv
        key = f"{args.problem}_{args.dtype}_nx{w.nx}_W{W}_{chain if chain else args.kernel}_nsteps{w.nsteps}"
        with open(os.path.join(ROOT, "profiles", "traffic.csv"), newline="") as f:
            for row in csv.DictReader(f):
                if row["key"] == key:
                    if row.get("kernel_sources_sha16", "") != kernel_sources_hash():
                        return None, f"stale: {row['report']} was captured from kernel sources {row.get('kernel_sources_sha16', '?')}, now {kernel_sources_hash()}"
                    return int(row["dram_bytes_per_launch"]), f"{row['report']} (kernel sources {row['kernel_sources_sha16']})"
    except Exception as e:
        return None, f"profiles/traffic.csv unreadable: {e}"
    return None, "no ncu --set full capture of this configuration under profiles/"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--problem", default="heat", choices=["heat", "ks", "euler"])
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--nx", type=int, default=1 << 22)
    ap.add_argument("--nsteps", type=int, default=0, help="timesteps per bench step (0 = the config's count)")
    ap.add_argument("--tile-width", type=int, default=0, help="0 = tuned (swept_tune)")
    ap.add_argument("--kernel", default="wave", choices=["wave", "smem"])
    ap.add_argument("--boundary", default="periodic", choices=["periodic", "insulated"],
                    help="insulated: the paper's own heat problem, a rod with insulated ends (heat only; SURVEY.md section 8(f) NEXT-2)")
    ap.add_argument("--sweep", action="store_true")
    ap.add_argument("--stress", action="store_true", help="BASELINE.json configs[4]: heat, KS, Euler x fp32, fp64 at nx = 2^22, 100 000 timesteps, "
                    "every tile width 32..2048 x kernel x resident-blocks cap 1..4 (written to gpurun_out/stress.json / stress.md)")
    ap.add_argument("--variants", default="", help="--sweep: comma list of ring,band,chain,wave,smem (default all)")
    ap.add_argument("--chain", type=int, default=3, choices=[0, 1, 2, 3],
                    help="launch-free sweep: 3 = ring kernel (default: bands + communication warp, remainder inside the launch), 2 = streaming bands, "
                         "1 = tile flags, 0 = one launch per half-cycle (PAPER.md:98)")
    ap.add_argument("--no-chain", action="store_true", help="same as --chain 0")
    ap.add_argument("--pack", type=int, default=0, choices=[0, 1, 2], help="SWEPT_OPT_PACK (heat fp32, band kernel): 0 auto / tuned, 1 off, 2 packed pairs of bands")
    ap.add_argument("--blocks-per-sm", type=int, default=0, help="SWEPT_OPT_BLOCKS_PER_SM for the per-tile kernels (0 = none / tuned)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-classic", action="store_true", help="skip the classic-path context run (profiling)")
    ap.add_argument("--no-range", action="store_true", help="skip the `sweep` points at nx = 2^11, 2^14, 2^17, 2^20 (profiling)")
    ap.add_argument("--probe", action="store_true", help="print the library's microbenchmarks as one JSON line: FP64 / FP32 FMA-chain peaks, shared-memory read peak, "
                    "latency probes (swept_measure_latencies): the denominators and bounds DESIGN.md quotes")
    ap.add_argument("--heat2d", action="store_true", help="secondary measurement (SURVEY.md section 8(f) NEXT-4): the 2-D swept rule against the classic "
                    "2-D kernel on an nx x nx periodic grid (--nx, default 8192; --nsteps, default 800), one JSON line")
    return ap.parse_args()


def workload_name(args, w) -> str:
    """config.workload: the same string on both arms (ours and --impl reference)."""
    if args.problem == "heat":
        return (f"BASELINE.json configs[1]: {w.name}, FTCS {args.boundary} r=0.25, nx=2^{int(np.log2(w.nx))}{' (largest of the sweep)' if w.nx == 1 << 22 else ''}, "
                f"{w.nsteps} timesteps per step")
    return f"{w.name} nx={w.nx} {w.nsteps} timesteps per step"


def workload(args) -> wl.Workload:
    w = wl.heat_rod(args.nx) if args.boundary == "insulated" else wl.make(args.problem, args.nx, "config")
    if args.boundary == "insulated":
        w.nsteps = 50_000                          # config 2's step count on the rod
    if args.nsteps:
        w.nsteps = args.nsteps
    return w


# ---------------------------------------------------------------------------------------------------------------
# ranks: "replicas only" -- every rank times its own replica; the job's time is the slowest rank's
# ---------------------------------------------------------------------------------------------------------------
def max_over_ranks(seconds: float, world: int, device="cpu") -> float:
    """MAX over ranks of a locally measured duration (the contract's max-over-ranks timing); no collective on the data path."""
    if world <= 1:
        return float(seconds)
    import torch
    import torch.distributed as dist
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(nx: int, nsteps: int, steps: int, world: int, t_max: float) -> float:
    """Whole-job GPts*steps/s: the units ALL ranks processed (world independent replicas) / the slowest rank's time."""
    return world * nx * nsteps * steps / t_max / 1e9


# ---------------------------------------------------------------------------------------------------------------
# clocks: sample nvidia-smi during the timed region (B200_PROFILING.md "clocks line")
# ---------------------------------------------------------------------------------------------------------------
class ClockSampler:
    """ONE long-lived `nvidia-smi -lms` process started before the timed region and read after it: no fork, no Python
    thread and no GIL traffic while the steps are being timed."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int, period_ms: int = 20):
        self.index, self.period_ms, self.rows, self._p = index, period_ms, [], None

    def __enter__(self):
        try:
            self._p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.index),
                                        "-lms", str(self.period_ms)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            time.sleep(0.3)          # let it attach and print its first rows before the timed region starts
        except Exception:
            self._p = None
        return self

    def __exit__(self, *exc):
        if self._p is None:
            return
        time.sleep(0.05)
        self._p.terminate()
        try:
            out, _ = self._p.communicate(timeout=5)
        except Exception:
            self._p.kill()
            out = ""
        for line in out.splitlines():
            cols = [c.strip() for c in line.split(",")]
            if len(cols) >= 7:
                self.rows.append(cols)

    def summary(self) -> dict:
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------------------
# CPU baseline / reference arm: the oracle as it stands, on the host cores, bounded sample
# ---------------------------------------------------------------------------------------------------------------
def oracle_rate(w: wl.Workload, dtype, budget_s: float = 15.0, insulated: bool = False):
    import oracle
    u0 = w.initial(dtype)
    kw = dict(dx=w.dx, dt=w.dt, alpha=w.alpha, gamma=w.gamma, insulated=insulated)
    oracle.run(w.problem, u0, 2, **kw)      # thread start-up, page faults
    t0 = time.perf_counter()
    oracle.run(w.problem, u0, 8, **kw)
    t8 = time.perf_counter() - t0
    n = int(max(8, min(w.nsteps, budget_s / max(t8 / 8, 1e-9))))
    t0 = time.perf_counter()
    oracle.run(w.problem, u0, n, **kw)
    dt = time.perf_counter() - t0
    # the same oracle on ONE thread (state both), about 3 s
    cores = oracle.num_threads()
    oracle.set_num_threads(1)
    try:
        n1 = int(max(2, min(n, 3.0 / max(t8 / 8 * cores, 1e-9))))      # one thread is at most `cores` times slower per step
        t0 = time.perf_counter()
        oracle.run(w.problem, u0, n1, **kw)
        rate1 = w.nx * n1 / (time.perf_counter() - t0)
    finally:
        oracle.set_num_threads(cores)
    return w.nx * n / dt, n, dt, cores, rate1


def run_reference(args):
    """--impl reference: this tier has no reference implementation; the reference arm is the CPU oracle."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = workload(args)
    dtype = np.float64 if args.dtype == "f64" else np.float32
    import oracle
    u0 = w.initial(dtype)
    okw = dict(dx=w.dx, dt=w.dt, alpha=w.alpha, gamma=w.gamma, insulated=args.boundary == "insulated")
    t0 = time.perf_counter()
    oracle.run(w.problem, u0, 2, **okw)
    per = (time.perf_counter() - t0) / 2
    total = max(1, args.steps + args.warmup)
    n = int(max(2, min(w.nsteps, (90.0 / total) / max(per, 1e-9))))    # whole run <= ~1.5 min
    for _ in range(args.warmup):
        oracle.run(w.problem, u0, n, **okw)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.run(w.problem, u0, n, **okw)
    el = time.perf_counter() - t0
    val = w.nx * n * args.steps / el / 1e9
    sample = f"{n} of the config's {w.nsteps} timesteps per step at nx={w.nx} (rate is step-count independent)"
    print(json.dumps({
        "impl": "reference", "metric": "grid-point updates/sec", "value": val, "unit": "GPts*steps/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": el / args.steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": workload_name(args, w), "arm": "CPU oracle (plain C, OpenMP) on the host cores, a bounded sample per step", "nx": w.nx,
                   "nsteps_per_step": n},
        "cpu_baseline": {"value": val, "unit": "GPts*steps/s", "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "GPts*steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ---------------------------------------------------------------------------------------------------------------
# --sweep: the paper's experiment E1/E2 (Fig. 8-9) re-measured on B200 -- for every nx of the config's
# range, every legal tile width against the classic path, best width kept.
# ---------------------------------------------------------------------------------------------------------------
SWEEP_NX = {"heat": range(11, 23), "ks": range(14, 21), "euler": range(12, 21)}


def metric_range(args, sizes=(11, 14, 17, 20)):
    """BASELINE.json's metric is quoted over nx = 2^11 ... 2^22 (the paper's experiment is the sweep, not one
    size).  The headline line times the largest size; this adds four more points of the same problem / dtype at the config's full
    step count -- the default swept path (swept_tune's choice, as in the headline) and the graph-launched classic path -- so that
    the driver's own run witnesses the range.  Each point: one warm-up call, then the median of 3 calls, CUDA events on the
    launching stream, L2 flushed between calls."""
    import torch

    import paper_1612_02495_b200 as sw

    np_dtype = np.float64 if args.dtype == "f64" else np.float32
    sw_dtype = sw.F64 if args.dtype == "f64" else sw.F32
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def timed(fn):
        fn()
        ts = []
        for _ in range(3):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); fn(); e1.record(stream); e1.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e-3)
        return statistics.median(ts)

    points = []
    for lg in sizes:
        nx = 1 << lg
        w = wl.make(args.problem, nx, "config")
        u0 = torch.from_numpy(w.initial(np_dtype)).cuda()
        u = u0.clone()
        with sw.Solver(w.problem, nx, w.dx, w.dt, dtype=sw_dtype, alpha=w.alpha, gamma=w.gamma) as s:
            W = s.tune(u.clone())
            t_swept = timed(lambda: s.swept_run(u, w.nsteps, W))
            info = s.info()
            kname = "smem" if info["tuned_kernel"] == sw.KERNEL_SMEM else sw.LAUNCH_NAMES.get(info["last_sweep_launch"], "?")
            launches = info["launches_last_call"]
            s.set_option(sw.OPT_NAIVE_GRAPH, 1)
            u.copy_(u0)
            t_classic = timed(lambda: s.naive_run(u, w.nsteps))
        points.append({"log2_nx": lg, "nsteps": w.nsteps, "swept": nx * w.nsteps / t_swept / 1e9, "tile_width": W, "kernel": kname,
                       "launches_per_run": int(launches), "classic_graph": nx * w.nsteps / t_classic / 1e9,
                       "speedup": t_classic / t_swept})
    return {"unit": "GPts*steps/s", "what": f"{args.problem} {args.dtype}, config step count, tuned swept path vs graph-launched classic path; "
                                            "median of 3 calls after a warm-up call, L2 flushed between calls", "points": points}


def run_sweep(args):
    import torch

    import paper_1612_02495_b200 as sw

    torch.cuda.set_device(0)
    np_dtype = np.float64 if args.dtype == "f64" else np.float32
    sw_dtype = sw.F64 if args.dtype == "f64" else sw.F32
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def timed(fn, reps=3):
        fn()                                   # warm-up (also builds a graph on first use)
        ts = []
        for _ in range(reps):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); fn(); e1.record(stream); e1.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e-3)
        return statistics.median(ts)

    rows = []
    for lg in SWEEP_NX[args.problem]:
        nx = 1 << lg
        w = wl.make(args.problem, nx, "config")
        if args.nsteps:
            w.nsteps = args.nsteps
        u0 = torch.from_numpy(w.initial(np_dtype)).cuda()
        u = u0.clone()
        row = {"nx": nx, "log2_nx": lg, "nsteps": w.nsteps, "swept": {}}
        with sw.Solver(w.problem, nx, w.dx, w.dt, dtype=sw_dtype, alpha=w.alpha, gamma=w.gamma) as s:
            ns_naive = min(w.nsteps, 2000)
            t = timed(lambda: s.naive_run(u, ns_naive))
            row["naive"] = nx * ns_naive / t / 1e9
            s.set_option(sw.OPT_NAIVE_GRAPH, 1)
            t = timed(lambda: s.naive_run(u, ns_naive))
            row["naive_graph"] = nx * ns_naive / t / 1e9
            # chain = launch-free sweep (one persistent launch); wave / smem = one launch per half-cycle, plain or CUDA graph
            for kname, kid, chain, graphs in (("ring", sw.KERNEL_WAVE, 3, (0,)), ("band", sw.KERNEL_WAVE, 2, (0,)), ("chain", sw.KERNEL_WAVE, 1, (0,)), ("wave", sw.KERNEL_WAVE, 0, (0, 1)),
                                              ("smem", sw.KERNEL_SMEM, 0, (0, 1))):
                if args.variants and kname not in args.variants.split(","):
                    continue
                s.set_option(sw.OPT_KERNEL, kid)
                s.set_option(sw.OPT_CHAIN, chain)
                for W in (32, 64, 128, 256, 512, 1024, 2048):
                    if W > nx or not s.tile_width_ok(W):
                        continue
                    for graph in graphs:
                        s.set_option(sw.OPT_SWEPT_GRAPH, graph)
                        u.copy_(u0)
                        t = timed(lambda: s.swept_run(u, w.nsteps, W), reps=3 if nx <= (1 << 20) else 2)
                        if kname in ("ring", "band") and sw.LAUNCH_NAMES.get(s.info()["last_sweep_launch"]) != kname:
                            continue                # the schedule does not fit this (nx, W): the run fell back, it is another row
                        row["swept"][f"{kname}/W={W}/{'graph' if graph else 'plain'}"] = nx * w.nsteps / t / 1e9
        best = max(row["swept"], key=row["swept"].get)
        row["best"], row["best_value"] = best, row["swept"][best]
        paper = [k for k in row["swept"] if k.startswith("smem") and k.endswith("plain")]
        best_paper = max(paper, key=row["swept"].get) if paper else best
        row["best_paper_style"], row["best_paper_style_value"] = best_paper, row["swept"][best_paper]
        row["speedup_vs_naive"] = row["best_value"] / row["naive"]
        row["speedup_vs_naive_graph"] = row["best_value"] / row["naive_graph"]
        rows.append(row)
        print(f"# nx=2^{lg}: naive {row['naive']:.2f} (graph {row['naive_graph']:.2f})  best swept {best} {row['best_value']:.1f} "
              f"GPts*steps/s  x{row['speedup_vs_naive']:.1f} / x{row['speedup_vs_naive_graph']:.1f}", file=sys.stderr, flush=True)
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    out = {"problem": args.problem, "dtype": args.dtype, "unit": "GPts*steps/s", "rows": rows}
    with open(os.path.join(ROOT, "gpurun_out", f"sweep_{args.problem}_{args.dtype}.json"), "w") as f:
        json.dump(out, f, indent=1)
    with open(os.path.join(ROOT, "gpurun_out", f"sweep_{args.problem}_{args.dtype}.csv"), "w") as f:      # the table profiles/sweeps/ keeps
        f.write("problem,dtype,log2_nx,nsteps,path,tile_width,launch,GPts_steps_per_s\n")
        for r in rows:
            f.write(f"{args.problem},{args.dtype},{r['log2_nx']},{r['nsteps']},classic,,plain,{r['naive']:.4f}\n")
            f.write(f"{args.problem},{args.dtype},{r['log2_nx']},{r['nsteps']},classic,,graph,{r['naive_graph']:.4f}\n")
            for k, v in r["swept"].items():
                kname, W, launch = k.split("/")
                f.write(f"{args.problem},{args.dtype},{r['log2_nx']},{r['nsteps']},{kname},{W[2:]},{launch},{v:.4f}\n")
    print(f"| nx | classic (plain launches) | classic (graph) | paper-style swept (smem, plain) | best swept | config | speedup vs classic | vs classic graph |")
    print("|---|---:|---:|---:|---:|---|---:|---:|")
    for r in rows:
        print(f"| 2^{r['log2_nx']} | {r['naive']:.2f} | {r['naive_graph']:.2f} | {r['best_paper_style_value']:.1f} ({r['best_paper_style'].split('/')[1]}) | "
              f"{r['best_value']:.1f} | {r['best']} | {r['speedup_vs_naive']:.1f}x | {r['speedup_vs_naive_graph']:.1f}x |")


# ---------------------------------------------------------------------------------------------------------------
# --stress: BASELINE.json configs[4] -- the tuning sweep at nx = 2^22
# ---------------------------------------------------------------------------------------------------------------
def run_stress(args):
    import torch

    import paper_1612_02495_b200 as sw

    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    nx = args.nx
    rows = []
    for problem in ("heat", "ks", "euler"):
        for dname in ("f64", "f32"):
            np_dtype = np.float64 if dname == "f64" else np.float32
            sw_dtype = sw.F64 if dname == "f64" else sw.F32
            w = wl.make(problem, nx, "config5")
            nsteps = args.nsteps or w.nsteps
            u0 = torch.from_numpy(w.initial(np_dtype)).cuda()
            u = u0.clone()

            def timed(fn):
                fn()
                flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream); fn(); e1.record(stream); e1.synchronize()
                return e0.elapsed_time(e1) * 1e-3

            with sw.Solver(w.problem, nx, w.dx, w.dt, dtype=sw_dtype, alpha=w.alpha, gamma=w.gamma) as s:
                ns_naive = min(nsteps, 1000)
                s.set_option(sw.OPT_NAIVE_GRAPH, 1)
                naive = nx * ns_naive / timed(lambda: s.naive_run(u, ns_naive)) / 1e9
                res = {}
                variants = [("ring", sw.KERNEL_WAVE, 3, (0,)), ("band", sw.KERNEL_WAVE, 2, (0,)), ("chain", sw.KERNEL_WAVE, 1, (0, 1, 2, 3, 4)),
                            ("smem", sw.KERNEL_SMEM, 0, (0, 1, 2, 3, 4))]
                if dname == "f32" and problem in ("heat", "ks"):
                    variants.insert(2, ("bandpack", sw.KERNEL_WAVE, 2, (0,)))     # the band kernel on packed f32x2 pairs (SWEPT_OPT_PACK = 2); "band" = one band per slot
                for kname, kid, chain, caps in variants:
                    s.set_option(sw.OPT_KERNEL, kid)
                    s.set_option(sw.OPT_CHAIN, chain)
                    s.set_option(sw.OPT_PACK, sw.PACK_ON if kname == "bandpack" else sw.PACK_OFF)
                    s.set_option(sw.OPT_SWEPT_GRAPH, 1 if kname == "smem" else 0)
                    for W in (32, 64, 128, 256, 512, 1024, 2048):
                        if not s.tile_width_ok(W):
                            continue
                        for cap in caps:
                            s.set_option(sw.OPT_BLOCKS_PER_SM, cap)
                            u.copy_(u0)
                            # rates do not depend on the step count: a 1000-step probe (also the warm-up) sizes the timed
                            # run to the config's 100 000 steps or about 1.5 s, whichever is shorter
                            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                            e0.record(stream); s.swept_run(u, 1000, W); e1.record(stream); e1.synchronize()
                            ns = int(min(nsteps, max(1000, 1000 * 1.5 / max(e0.elapsed_time(e1) * 1e-3, 1e-6))))
                            u.copy_(u0)
                            flush.zero_()
                            e0.record(stream); s.swept_run(u, ns, W); e1.record(stream); e1.synchronize()
                            t = e0.elapsed_time(e1) * 1e-3
                            ran = sw.LAUNCH_NAMES.get(s.info()["last_sweep_launch"], "-") if kname != "smem" else "smem"
                            if kname in ("ring", "band", "bandpack") and ran != kname.replace("pack", ""):
                                continue            # the schedule does not fit: this (W) is another kernel's row
                            res[f"{kname}/W={W}/cap={cap}"] = nx * ns / t / 1e9
                s.set_option(sw.OPT_BLOCKS_PER_SM, 0)
            best = max(res, key=res.get)
            rows.append({"problem": problem, "dtype": dname, "nx": nx, "nsteps": nsteps, "classic_graph": naive, "results": res, "best": best,
                         "best_value": res[best]})
            print(f"# {problem} {dname}: classic(graph) {naive:.1f}  best {best} {res[best]:.1f} GPts*steps/s", file=sys.stderr, flush=True)
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    with open(os.path.join(ROOT, "gpurun_out", "stress.json"), "w") as f:
        json.dump({"unit": "GPts*steps/s", "rows": rows}, f, indent=1)
    with open(os.path.join(ROOT, "gpurun_out", "stress_config5.csv"), "w") as f:
        f.write("problem,dtype,nx,nsteps,path,tile_width,blocks_per_sm_cap,GPts_steps_per_s\n")
        for r in rows:
            f.write(f"{r['problem']},{r['dtype']},{r['nx']},{r['nsteps']},classic(graph),,,{r['classic_graph']:.4f}\n")
            for k, v in r["results"].items():
                kname, W, cap = k.split("/")
                f.write(f"{r['problem']},{r['dtype']},{r['nx']},{r['nsteps']},{kname},{W[2:]},{cap[4:]},{v:.4f}\n")
    print("| problem | dtype | classic (graph) | best swept | config | x classic | best per kernel: ring | band (one band per slot) | band, packed pairs | chain (W, cap) | smem (W, cap) |")
    print("|---|---|---:|---:|---|---:|---|---|---|---|---|")
    for r in rows:
        def bk(k):
            c = {n: v for n, v in r["results"].items() if n.startswith(k + "/")}
            if not c:
                return "-"
            b = max(c, key=c.get)
            return f"{c[b]:.1f} ({b.split('/', 1)[1]})"
        print(f"| {r['problem']} | {r['dtype']} | {r['classic_graph']:.1f} | {r['best_value']:.1f} | {r['best']} | {r['best_value'] / r['classic_graph']:.1f}x | "
              f"{bk('ring')} | {bk('band')} | {bk('bandpack')} | {bk('chain')} | {bk('smem')} |")


def run_heat2d(args):
    """2-D heat, fp64 / fp32, nx x nx (HBM-resident at the default 8192^2 = 512 MiB): swept (W = 32, 16) vs classic, CUDA-event timed."""
    import torch

    import paper_1612_02495_b200 as sw

    torch.cuda.set_device(0)
    n = args.nx if args.nx != (1 << 22) else 8192
    nsteps = args.nsteps or 800
    np_dtype = np.float64 if args.dtype == "f64" else np.float32
    dx, dt = wl.heat2d_grid(n, 0.2)
    u0 = torch.from_numpy(wl.heat2d_field(n, n).astype(np_dtype)).cuda()
    u = u0.clone()
    stream = torch.cuda.current_stream()

    def timed(fn):
        fn()
        ts = []
        for _ in range(max(args.steps, 3)):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); fn(); e1.record(stream); e1.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e-3)
        return statistics.median(ts)

    res = {}
    with sw.Solver2D(n, n, dx, dt, dtype=sw.F64 if args.dtype == "f64" else sw.F32) as s:
        t = timed(lambda: s.naive_run(u, nsteps))
        res["classic"] = n * n * nsteps / t / 1e9
        for W, kern, kname in ((32, sw.KERNEL2D_WARP, "register kernel"), (32, sw.KERNEL2D_COLUMN, "register kernel, one column per lane"), (32, sw.KERNEL2D_SMEM, "paper-style smem kernel"), (16, sw.KERNEL2D_SMEM, "paper-style smem kernel"),
                               (8, sw.KERNEL2D_SMEM, "paper-style smem kernel")):
            s.set_option(sw.OPT2D_KERNEL, kern)
            u.copy_(u0)
            t = timed(lambda: s.swept_run(u, nsteps, W))
            res[f"swept W={W} ({kname})"] = n * n * nsteps / t / 1e9
        # e2e: the same run through swept2d_run_host -- H2D of the field from pinned host memory, the default swept path (register
        # kernel, W = 32), D2H of the result, synchronise -- wall-clock around the C-ABI call, median of 3
        s.set_option(sw.OPT2D_KERNEL, sw.KERNEL2D_WARP)
        h_u = u0.cpu().pin_memory()
        s.run_host(h_u, nsteps, 32)
        ts = []
        for _ in range(3):
            h_u.copy_(u0)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            s.run_host(h_u, nsteps, 32)
            ts.append(time.perf_counter() - t0)
        e2e_val = n * n * nsteps / statistics.median(ts) / 1e9
    try:
        hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
        hbm_src = "measured (MEASURED_PEAKS.json)"
    except Exception:
        hbm_peak, hbm_src = 6650.0, "fallback (B200_PROFILING.md)"
    es = u.element_size()
    best = max((k for k in res if k.startswith("swept")), key=res.get)
    Wb = int(best.split("W=")[1].split()[0])
    # roofline of the swept path: by algorithmic bytes it would be HBM-bound (7 values per point per half-cycle of W/2 timesteps, see
    # below), by arithmetic FP-pipe-bound (5 FP instructions per update: 3 adds, 1 multiply, 1 fma); it reaches neither (DESIGN.md
    # section 5.8: issue- and latency-bound at 8 warps per SM), so both fractions are stated and `bound` names the nearer one
    bytes_per_update = 7 * es / (Wb // 2)
    hbm_frac = res[best] * bytes_per_update / hbm_peak
    alu_peak = 148 * (64 if args.dtype == "f64" else 128) * 1.965e-3          # T thread-level FP instr/s, nominal pipe
    alu_frac = res[best] * 5e-3 / alu_peak
    cpu = None
    if not args.no_cpu_baseline:
        import oracle
        a0 = wl.heat2d_field(n, n).astype(np_dtype)
        oracle.heat2d(a0, 1, 1.0, dx, dt)
        t0 = time.perf_counter(); oracle.heat2d(a0, 4, 1.0, dx, dt); t4 = time.perf_counter() - t0
        k = int(max(4, min(nsteps, 12.0 / max(t4 / 4, 1e-9))))
        t0 = time.perf_counter(); oracle.heat2d(a0, k, 1.0, dx, dt); el = time.perf_counter() - t0
        cpu = {"value": n * n * k / el / 1e9, "unit": "GPts*steps/s", "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"{k} of {nsteps} timesteps at {n} x {n} ({el:.1f} s)"}
    print(json.dumps({
        "metric": "grid-point updates/sec (2-D heat, secondary)", "unit": "GPts*steps/s", "value": res[best], "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": f"2-D heat FTCS 5-point, periodic {n} x {n}, Fo = 0.2, {nsteps} timesteps; field {n * n * es >> 20} MiB (larger than L2)", "best": best},
        "results": res, "speedup_swept_over_classic": res[best] / res["classic"],
        "e2e": {"value": e2e_val, "unit": "GPts*steps/s", "h2d_bytes_per_step": n * n * es, "d2h_bytes_per_step": n * n * es,
                "what": "swept2d_run_host, register kernel W = 32, pinned host buffer, wall clock around the call, median of 3"},
        "roofline": {"bound": "hbm" if hbm_frac >= alu_frac else "alu", "kernel": best, "achieved": res[best] * bytes_per_update, "peak": hbm_peak, "unit": "GB/s",
                     "frac": hbm_frac, "peak_source": hbm_src, "algorithmic_bytes_per_update": bytes_per_update,
                     "alu_frac": alu_frac, "alu_peak_Tinstr_s": alu_peak, "fp_instr_per_update": 5,
                     "traffic": None, "traffic_source": "profiles/r2_ncu_2d_warp.md: 1.27 GB of DRAM traffic per half-cycle at 8192^2 fp64 = 4.7 B per update, 1.34 x the algorithmic 3.5 B"},
        "cpu_baseline": cpu,
        "classic_roofline": {"bound": "hbm", "algorithmic_bytes_per_update": 2 * es, "achieved_GBps": res["classic"] * 2 * es, "peak_GBps": hbm_peak,
                             "frac": res["classic"] * 2 * es / hbm_peak},
        # swept: per half-cycle of L = W/2 timesteps the two launches (bridges, octahedra) each read both arrays over every tile
        # box and write what they updated: about 4 reads + 3 writes per point = 7 values per L timesteps
        "swept_hbm_algorithmic_bytes_per_update": {f"W={W}": 7 * es / (W // 2) for W in (32, 16, 8)},
    }))


def main():
    args = parse()
    if args.probe:
        import torch
        import paper_1612_02495_b200 as sw
        torch.cuda.set_device(0)
        print(json.dumps({"alu_peak_f64_Tinstr_s": sw.measure_alu_peak(sw.F64)["instr_per_s"] / 1e12, "alu_peak_f32_Tinstr_s": sw.measure_alu_peak(sw.F32)["instr_per_s"] / 1e12,
                          "nominal_f64_Tinstr_s": 148 * 64 * 1.965e-3, "nominal_f32_Tinstr_s": 148 * 128 * 1.965e-3,
                          "smem_peak_GBps": sw.measure_smem_peak()["bytes_per_s"] / 1e9, "smem_nominal_GBps": 148 * 128 * 1.965,
                          "latency_cycles": sw.measure_latencies()}))
        return
    if args.heat2d:
        run_heat2d(args)
        return
    if args.impl == "reference":
        run_reference(args)
        return
    if args.sweep:
        run_sweep(args)
        return
    if args.stress:
        run_stress(args)
        return

    import torch
    import torch.distributed as dist

    import paper_1612_02495_b200 as sw

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the swept path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    w = workload(args)
    np_dtype = np.float64 if args.dtype == "f64" else np.float32
    sw_dtype = sw.F64 if args.dtype == "f64" else sw.F32
    kernel = sw.KERNEL_WAVE if args.kernel == "wave" else sw.KERNEL_SMEM
    s = sw.Solver(w.problem, w.nx, w.dx, w.dt, dtype=sw_dtype, alpha=w.alpha, gamma=w.gamma,
                  boundary=sw.BC_INSULATED if args.boundary == "insulated" else sw.BC_PERIODIC)
    s.set_option(sw.OPT_KERNEL, kernel)
    chain_opt = 0 if args.no_chain else args.chain
    s.set_option(sw.OPT_CHAIN, chain_opt)
    if args.blocks_per_sm:
        s.set_option(sw.OPT_BLOCKS_PER_SM, args.blocks_per_sm)
    if args.pack:
        s.set_option(sw.OPT_PACK, args.pack)
    if not any(s.tile_width_ok(W) for W in (32, 64, 128, 256, 512, 1024)):
        kernel = sw.KERNEL_SMEM
        s.set_option(sw.OPT_KERNEL, kernel)
    u0_host = torch.from_numpy(w.initial(np_dtype)).pin_memory()
    u = u0_host.cuda()
    stream = torch.cuda.current_stream()
    t_tune0 = time.perf_counter()
    W = args.tile_width or s.tune(u.clone())
    torch.cuda.synchronize()
    tune_ms = (time.perf_counter() - t_tune0) * 1e3 if not args.tile_width else 0.0      # wall time of swept_tune (outside the timed region)
    tune_launches = s.info()["launches_total"]
    if not args.tile_width and s.info()["tuned_kernel"] == sw.KERNEL_SMEM:
        kernel = sw.KERNEL_SMEM                   # the tuner measured the paper-style kernels as fastest (small Euler grids): swept_run follows it
    sph = sw.steps_per_half_cycle(w.problem, W)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, k):
        """k calls of fn, each bracketed by CUDA events on the launching stream, L2 flushed between calls."""
        tot = 0.0
        for _ in range(k):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            fn()
            e1.record(stream)
            e1.synchronize()
            tot += e0.elapsed_time(e1) * 1e-3
        return tot

    # ---- device-resident timing: inputs already in HBM ----------------------------------------------------
    def step_dev():
        s.swept_run(u, w.nsteps, W)

    for _ in range(max(args.warmup, 3)):
        u.copy_(u0_host, non_blocking=True)
        step_dev()
    barrier()
    l0 = s.info()["launches_total"]
    with ClockSampler(local_rank) as clk:
        barrier()
        t_dev = timed(step_dev, args.steps)
        barrier()
    launches = s.info()["launches_total"] - l0
    t_dev_max = max_over_ranks(t_dev, world, "cuda")
    value = job_value(w.nx, w.nsteps, args.steps, world, t_dev_max)

    # ---- end to end through the C ABI with HOST buffers (H2D + D2H inside the timed region) ----------------
    h_buf = u0_host.clone().pin_memory()

    def step_e2e():
        s.run_host(h_buf, w.nsteps, W, use_swept=True)

    step_e2e()
    barrier()
    t_e2e = timed(step_e2e, args.steps)
    e2e_value = job_value(w.nx, w.nsteps, args.steps, world, max_over_ranks(t_e2e, world, "cuda"))
    field_bytes = int(u.numel() * u.element_size())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel -------------------------------------------------------------------
    # launch-free kernels: ONE launch runs the sweep.  ring (default): the whole step -- q half-cycles and the remainder -- is that
    # launch, nx * S * nsteps stage-updates.  band / tile flags: q half-cycles = nx * L * q stage-updates, timed alone (nsteps = q * sph
    # has no remainder, so the plan is that single launch + the memset of its flags).
    # per-launch kernels (--chain 0 / smem): the diamond launch, by differencing two runs of qa and qb half-cycles.
    pinfo = sw.problem_info(w.problem)
    H, S = pinfo["radius"], pinfo["stages"]
    L = W // (2 * H)
    chain = kernel == sw.KERNEL_WAVE and chain_opt != 0
    step_kind = s.info()["last_sweep_launch"]           # what the timed steps ran on
    q = max(1, w.nsteps // sph)
    if chain and step_kind == sw.LAUNCH_RING:
        assert sw.plan(w.problem, w.nx, w.nsteps, W, dtype=sw_dtype, chain=chain_opt) == [(sw.LAUNCH_RING, W, w.nsteps % sph, w.nsteps // sph)]
        run_q = lambda: s.swept_run(u, w.nsteps, W)
        run_q()
        t_launch = min(timed(run_q, 1) for _ in range(3))
        stage_updates = w.nx * S * w.nsteps
        lname = "ring"
        kname = f"swept_ring_kernel W={W} ({w.nsteps // sph} half-cycles + {w.nsteps % sph} remainder timesteps in one launch)"
        hc = w.nsteps / sph
    elif chain:
        run_q = lambda: s.swept_run(u, q * sph, W)
        run_q()
        t_launch = min(timed(run_q, 1) for _ in range(3))
        stage_updates = w.nx * L * q
        lname = {sw.LAUNCH_BAND: "band", sw.LAUNCH_RING: "ring"}.get(s.info()["last_sweep_launch"], "chain")
        kname = f"swept_{lname}_kernel W={W} ({q} half-cycles in one launch)"
        hc = q
    else:
        def half_cycles(n):
            return lambda: s.swept_run(u, n * sph, W)
        qa, qb = 16, 48
        for n in (qa, qb):
            half_cycles(n)()
        ta = min(timed(half_cycles(qa), 1) for _ in range(3))
        tb = min(timed(half_cycles(qb), 1) for _ in range(3))
        t_launch = (tb - ta) / (qb - qa)
        stage_updates = w.nx * L                               # per diamond launch: every point advances L tiers
        lname = ""
        kname = f"swept diamond ({'wave' if kernel == sw.KERNEL_WAVE else 'smem'}) W={W}"
        hc = 1
    band = lname in ("band", "ring")
    fpi = FP_INSTR_PER_STAGE_UPDATE[(args.problem, args.dtype)]
    peak_meas = sw.measure_alu_peak(sw_dtype)["instr_per_s"]
    nominal = 148 * (64 if args.dtype == "f64" else 128) * 1.965e9
    achieved = fpi * stage_updates / t_launch if fpi else None
    traffic, traffic_source = traffic_of(args, w, W, lname)
    roofline = {
        "bound": "alu", "kernel": kname,
        "achieved": achieved / 1e12 if achieved else None, "peak": nominal / 1e12, "unit": "T FP-instr/s (thread-level)",
        "frac": (achieved / nominal) if achieved else None,
        "peak_source": "nominal pipe: 148 SMs x %d lanes x 1.965 GHz (DESIGN.md section 5.3; MEASURED_PEAKS.json has no plain-ALU figure)" % (64 if args.dtype == "f64" else 128),
        "peak_measured_alu": peak_meas / 1e12, "frac_measured_alu": (achieved / peak_meas) if achieved else None,
        "peak_measured_alu_source": "FMA-chain microbenchmark (swept_measure_alu_peak), same process, same clocks",
        "traffic": traffic, "traffic_source": traffic_source,
        "launch_ms": t_launch * 1e3, "fp_instr_per_stage_update": fpi, "stage_updates_per_launch": stage_updates,
        # staircase bytes: per half-cycle every tile reads and writes both edges (4 W values), the band / ring kernels only the
        # upper-right edge (2 W values: lane 31's row outputs out, lane 0's row feed in)
        "hbm_algorithmic_bytes_per_launch": int((2 if band else 4) * w.nx * pinfo["ncomp"] * u.element_size() * hc),
    }
    # shared-memory roofline (north_star: "shared-memory throughput for the swept path ... against the chip's peak"): it bounds the
    # paper-style kernels, which move (2h + 1) loads + 1 store of shared memory per point update; the register kernels touch
    # shared memory only for the edge rings (2 s / PW bytes per update and less)
    smem_peak = sw.measure_smem_peak()["bytes_per_s"]
    roofline["smem_peak_measured_GBps"] = smem_peak / 1e9
    roofline["smem_peak_nominal_GBps"] = 148 * 128 * 1.965
    if kernel == sw.KERNEL_SMEM:
        smem_bytes = (2 * H + 2) * pinfo["ncomp"] * u.element_size() * stage_updates
        roofline["smem_achieved_GBps"] = smem_bytes / t_launch / 1e9
        roofline["smem_frac"] = smem_bytes / t_launch / smem_peak
        roofline["bound"] = "smem"

    # ---- classic path on the same workload (context: swept / classic speedup) ------------------------------
    classic = None
    if not args.no_classic:
        ns_naive = min(w.nsteps, 2000)
        u.copy_(u0_host)
        s.naive_run(u, ns_naive)
        t_naive = timed(lambda: s.naive_run(u, ns_naive), 1)
        naive_val = w.nx * ns_naive / t_naive / 1e9
        s.set_option(sw.OPT_NAIVE_GRAPH, 1)
        s.naive_run(u, ns_naive)
        t_naive_g = timed(lambda: s.naive_run(u, ns_naive), 1)
        naive_graph_val = w.nx * ns_naive / t_naive_g / 1e9
        shared_val = None
        if args.problem == "euler":               # the classic kernel with the faces between a thread's cells evaluated once (SWEPT_OPT_NAIVE_SHARE)
            s.set_option(sw.OPT_NAIVE_SHARE, 1)
            s.naive_run(u, ns_naive)
            shared_val = w.nx * ns_naive / timed(lambda: s.naive_run(u, ns_naive), 1) / 1e9
            s.set_option(sw.OPT_NAIVE_SHARE, 0)
        naive_bytes = {"heat": 2, "ks": 5, "euler": 15}[args.problem] * u.element_size()
        try:
            hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
            hbm_src = "measured (MEASURED_PEAKS.json)"
        except Exception:
            hbm_peak, hbm_src = 6650.0, "fallback (B200_PROFILING.md)"
        classic = {"value": naive_val, "value_graph": naive_graph_val, "value_graph_shared_faces": shared_val, "unit": "GPts*steps/s", "timesteps": ns_naive,
                   "algorithmic_GBps": naive_val * naive_bytes, "algorithmic_GBps_graph": naive_graph_val * naive_bytes,
                   "hbm_peak_GBps": hbm_peak, "hbm_peak_source": hbm_src,
                   "frac_of_hbm": max(naive_val, naive_graph_val) * naive_bytes / hbm_peak,
                   "note": "fields up to nx=2^22 are L2-resident, so the classic path can exceed the HBM figure",
                   "speedup_swept_over_classic": value / world / max(naive_val, naive_graph_val)}

    cpu = None
    if not args.no_cpu_baseline:
        rate, n, el, cores, rate1 = oracle_rate(w, np_dtype, insulated=args.boundary == "insulated")
        cpu = {"value": rate / 1e9, "unit": "GPts*steps/s", "cores": cores, "kind": "oracle", "value_1_thread": rate1 / 1e9,
               "sample": f"{n} of {w.nsteps} timesteps at nx={w.nx} ({el:.1f} s)"}

    sweep = None
    if rank == 0 and world == 1 and not (args.no_range or args.no_classic) and args.boundary == "periodic":
        sweep = metric_range(args)

    out = {
        "metric": "grid-point updates/sec", "value": value, "unit": "GPts*steps/s", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": t_dev_max / args.steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
        "config": {
            "workload": workload_name(args, w),
            "nx": w.nx, "nsteps_per_step": w.nsteps, "boundary": args.boundary, "tile_width": W,
            "kernel": (lname if chain else "wave") if kernel == sw.KERNEL_WAVE else "smem",
            "tile_width_source": "--tile-width" if args.tile_width else "swept_tune, before the timed region",
            "tune_ms": tune_ms, "tune_launches": int(tune_launches), "tuned_pack": s.info()["tuned_pack"],
            "parallelism": "replicas only" if world > 1 else "1 GPU",
            "l2": "L2 flushed (256 MB write) between timed steps; the 32 MiB field is L2-resident within a step by the config's size",
        },
        "e2e": {"value": e2e_value, "unit": "GPts*steps/s", "h2d_bytes_per_step": field_bytes, "d2h_bytes_per_step": field_bytes},
        "gpu_launches": int(launches),
        "clocks": clk.summary(),
        "roofline": roofline,
        "cpu_baseline": cpu,
        "classic": classic,
        "sweep": sweep,
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
