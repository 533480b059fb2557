#!/usr/bin/env python
"""bench.py -- GFCCSD-IP hot path on B200: sigma-matvec FP64 TFLOP/s and (p,omega) solves/s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]
    torchrun --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...      (one rank per GPU)

A STEP is one pass of the whole hot path over one batch of synthetic right-hand sides: one gfcc_solve_ip call
in fixed-iteration mode (gmres_fixed = KFIX Arnoldi steps => KFIX+1 batched sigma applications S1-S13, the
CGS2/Givens work G1-G5 and the G_pq assembly G6).  The one-time intermediates (gfcc_create, P1-P7, PAPER.md:173
"pre-computed before entering the main GFCC loop") are built before the timed region and reported as create_s.
`value` = (KFIX+1) * F_sigma / step time: sigma FP64 TFLOP/s of the WHOLE step (GMRES and G time are charged
against it); F_sigma is the executed flop model of SURVEY.md 8(d) (real x complex counted as 2 real products,
pair-packed o^4 term).  N > 1: the (p,omega) list is sharded over ranks (independent tasks),
no data-path collective, weak scaling.

Inputs are seeded and synthetic (gfcc_inputs) and stand in for the paper's molecular
workloads.  The working set of every config >= 1 is far larger than the 126 MB L2.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

FP64_DMMA_PEAK_R1 = 36.95       # round-1 value of the DMMA.8x8x4 issue-rate probe (profiles/fp64_peak_probe.md); the probe is re-run in every bench run
KFIX = {0: 20, 1: 8, 2: 20, 3: 2, 4: 1}     # Arnoldi steps per timed step (config 2: BASELINE.json "20 GMRES iterations fixed for timing";
                                            # configs 3-4 bounded so that a default run ends in minutes: one step is 39 s at config 4)
DEFAULT_CONFIG = 4
NCU_TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r2_gemm_ncu_traffic.csv")   # ncu --set full captures of the step's GEMM launches


def ncu_traffic(cfg):
    """DRAM bytes of the dominant launch shape of a config-`cfg` step, read from the tracked ncu summary (never a constant
    in this file): the row of NCU_TRAFFIC_CSV with this config whose `dominant` column is 1."""
    try:
        import csv
        with open(NCU_TRAFFIC_CSV) as f:
            for row in csv.DictReader(l for l in f if not l.startswith("#")):
                if int(row["config"]) == cfg and int(row["dominant"]) == 1:
                    return {"bytes": float(row["dram_read_bytes"]) + float(row["dram_write_bytes"]), "launch": row["launch"],
                            "shape": f"{row['M']} x {row['N']} x {row['K']} (BM = {row['BM']})",
                            "algorithmic_bytes": float(row["algorithmic_bytes"]), "source": os.path.relpath(NCU_TRAFFIC_CSV, ROOT)}
    except Exception:
        pass
    return None


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kfix", type=int, default=0, help="Arnoldi steps per step (default: per config)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-solves", action="store_true", help="skip the converged-solve rate measurement (config 0 and config 1)")
    ap.add_argument("--cpu-baseline-only", action="store_true",
                    help="(internal) child process of the default run: time the oracle sample, print its JSON, exit")
    ap.add_argument("--cpu-baseline-serial", action="store_true",
                    help="time the oracle AFTER the GPU part on all host cores instead of beside it (doubles the run time at config 4)")
    ap.add_argument("--engine", default="dmma", choices=["dmma", "ozaki"],
                    help="dmma: FP64 tensor-core engine (graded default); ozaki: S8-S11 on the INT8 tensor pipe with FP64 accuracy "
                         "(SURVEY.md 8f row 2, reported separately)")
    ap.add_argument("--slices", type=int, default=7, help="digit slices of the ozaki engine (7: ~1e-13, 6: ~1e-11 per GEMM)")
    ap.add_argument("--no-ozaki-extra", action="store_true", help="skip the extra INT8-engine measurement appended to a dmma run")
    ap.add_argument("--panel-bytes", type=float, default=0.0, help="byte budget of one (ov x ov) integral panel (default: library default)")
    ap.add_argument("--overlap", type=int, default=-1, help="1: run independent sigma panel chains on side streams (default: library default)")
    return ap.parse_args()


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return None


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""

    def __init__(self, gpu_index):
        super().__init__(daemon=True)
        self.gpu = gpu_index
        self.samples, self.reasons, self.maxclk = [], set(), None
        self.stop_flag = False

    def run(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i", str(self.gpu)],
                                     capture_output=True, text=True, timeout=5).stdout.strip().split(",")
                self.samples.append(float(out[0]))
                self.maxclk = float(out[1])
                for n, val in zip(names, out[2:]):
                    if "Active" in val and "Not" not in val:
                        self.reasons.add(n)
            except Exception:
                pass
            time.sleep(0.2)

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.maxclk, "reasons": sorted(self.reasons),
                "samples": len(s)}


def workload_string(cfg, c, nrhs, kfix, rank_shift):
    return (f"config{cfg}: o={c['o']} v={c['v']} Q={c['Q']} nrhs={nrhs} ({c['np']} p x {c['nw']} omega per GPU), eta={c['eta']}, "
            f"one gfcc_solve_ip with {kfix} fixed Arnoldi steps = {kfix + 1} batched sigma applications + CGS2/Givens + G assembly")


# ---------------------------------------------------------------------------------------------------------
def oracle_sample(cfg, c, nrhs_s, ns_small, ns_large, ready_cb=None):
    """time the CPU oracle (as it stands) on a bounded sample of the workload: the row-sampled sigma at TWO sample sizes
    (ns_small and ns_large sigma2 rows, each with one sigma1 row and nrhs_s right-hand sides) so that the per-call part
    (Y, yv over the whole vector) can be separated from the per-row part."""
    import torch
    import gfcc_inputs as gi
    import oracle
    o, v, Q = c["o"], c["v"], c["Q"]
    dev = "cuda" if (torch.cuda.is_available() and cfg >= 2) else "cpu"
    s = gi.make_config(cfg, dev)
    host = {k: s[k].cpu().numpy() for k in ("fock", "T1", "T2p", "L1", "L2p", "Lchol")}
    X1, X2 = gi.trial_vectors(o, v, nrhs_s, gi.seed_of(cfg), dev)
    X1, X2 = X1.cpu().numpy(), X2.cpu().numpy()
    del s
    if dev == "cuda":
        torch.cuda.empty_cache()
    if ready_cb is not None:
        ready_cb()
    w = np.linspace(c["wlo"], c["whi"], nrhs_s)
    t0 = time.time()
    orc = oracle.Oracle(o, v, Q, host["fock"], host["T1"], host["T2p"], host["L1"], host["L2p"], host["Lchol"], oracle.MODE_ROWS)
    t_setup = time.time() - t0
    rng = np.random.default_rng(7)
    times = []
    for ns in (ns_small, ns_large):
        trip = np.stack([rng.integers(0, o - 1, ns), np.full(ns, o - 1), rng.integers(0, v, ns)], axis=1)
        t0 = time.time()
        orc.sigma_rows(w, c["eta"], X1, X2, [o - 1], trip)
        times.append(time.time() - t0)
    return t_setup, times, oracle.threads()


def cpu_baseline(cfg, c, nrhs, flops_sigma, ready_cb=None):
    """bounded oracle sample -> extrapolated seconds for ONE batched sigma application of the oracle as it stands:
    t(ns rows, nrhs_s RHS) = t_call + ns * t_row is fitted to the two timings; a full application is one call with all
    npair*v rows and nrhs RHS: t_call * (nrhs / nrhs_s) + npair * v * t_row (the row part does not grow with the number of
    right-hand sides to first order: the row-sampled routine rebuilds O(o^2 v Q) intermediates per row, which is what makes it a
    checker and not a sigma implementation -- the number is a baseline, not a target)."""
    nrhs_s = 2
    ns_small, ns_large = (2, 10) if cfg <= 2 else ((1, 4) if cfg == 3 else (1, 2))   # ~65 s per sigma2 row at config 4
    t_setup, (t_a, t_b), cores = oracle_sample(cfg, c, nrhs_s, ns_small, ns_large, ready_cb)
    t_row = max((t_b - t_a) / (ns_large - ns_small), 1e-9)
    t_call = max(t_a - ns_small * t_row, 0.0)
    npair = c["o"] * (c["o"] - 1) // 2
    rows_total = npair * c["v"]
    t_full = t_call * (nrhs / nrhs_s) + rows_total * t_row
    return {"seconds_full": t_full, "value": flops_sigma / t_full / 1e12, "unit": "TFLOP/s", "cores": cores, "kind": "oracle",
            "sample": (f"row-sampled oracle sigma (oracle/gfcc_oracle.cpp orc_sigma_rows) of config {cfg} at two sample sizes: "
                       f"{ns_small} and {ns_large} sigma2 rows (+1 sigma1 row) x {nrhs_s} RHS in {t_a:.1f} s and {t_b:.1f} s -> per-call part "
                       f"{t_call:.1f} s, per-row part {t_row:.2f} s (one-time dressing {t_setup:.1f} s, not charged); one batched application = "
                       f"{rows_total} rows x {nrhs} RHS in one call: EXTRAPOLATED by a factor {rows_total / ns_large:.3g} in the row count"),
            "seconds_per_row": t_row, "seconds_per_call": t_call, "seconds_setup": t_setup, "extrapolation_factor": rows_total / ns_large}


def model_flops(c, nrhs):
    """executed flop model of one batched sigma application; the library reports the same
    number as gfcc_get_stat(h, "flops_sigma")."""
    o, v, Q = c["o"], c["v"], c["Q"]
    npair = o * (o - 1) // 2
    Nc = 2.0 * nrhs
    ov = o * v
    return (2 * Q * ov * o * Nc * 2 + 4 * Q * ov * ov + 6 * ov * ov * o * Nc + 2 * npair * npair * v * Nc
            + 2 * npair * v * v * Nc + 2 * npair * v * o * Nc + 2 * Q * o * v * Nc + 2 * Q * o * o * Nc + 2 * ov * o * Nc)


def run_cpu_baseline_child(args):
    """child of the default run: generates its own copy of the inputs (on the GPU when there is one, then moved to the
    host and the device memory released), prints READY, times the oracle sample, prints one JSON line."""
    import gfcc_inputs as gi
    c = gi.CONFIGS[args.config]
    nrhs = c["np"] * c["nw"]
    cb = cpu_baseline(args.config, c, nrhs, model_flops(c, nrhs), ready_cb=lambda: print("READY", flush=True))
    print(json.dumps(cb), flush=True)
    return 0


def start_cpu_baseline_child(cfg):
    """start the oracle timing in a child process on ALL host cores.  It overlaps only the untimed GPU phases of this run (input
    generation, gfcc_create, warm-up): main() waits for it BEFORE the timed region starts, so neither measurement disturbs the other."""
    child = subprocess.Popen([sys.executable, os.path.abspath(__file__), "--cpu-baseline-only", "--config", str(cfg)],
                             stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True, env=dict(os.environ))
    while True:                                   # wait until the child has released the device memory of its inputs
        ln = child.stdout.readline()
        if not ln or ln.strip() == "READY":
            break
    return child


def finish_cpu_baseline_child(child, flops_sigma, timeout_s=1800):
    try:
        out, _ = child.communicate(timeout=timeout_s)
    except subprocess.TimeoutExpired:
        child.kill()
        return {"value": None, "unit": "TFLOP/s", "cores": None, "kind": "oracle", "sample": f"oracle sample not finished after {timeout_s} s"}
    for ln in reversed(out.strip().splitlines()):
        if ln.startswith("{"):
            cb = json.loads(ln)
            cb["value"] = flops_sigma / cb.pop("seconds_full") / 1e12
            cb["sample"] += "; timed in a child process on all host cores during input generation / gfcc_create / warm-up, finished before the timed region"
            return cb
    return {"value": None, "unit": "TFLOP/s", "cores": None, "kind": "oracle", "sample": "oracle child printed no result"}


# ---------------------------------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import gfcc_inputs as gi
    cfg = args.config
    c = gi.CONFIGS[cfg]
    nrhs = c["np"] * c["nw"]
    kfix = args.kfix or KFIX[cfg]
    o, v, Q = c["o"], c["v"], c["Q"]
    npair = o * (o - 1) // 2
    flops_sigma = model_flops(c, nrhs)
    vals = []
    last = None
    for it in range(args.warmup + args.steps):
        cb = cpu_baseline(cfg, c, nrhs, flops_sigma)
        if it >= args.warmup:
            vals.append(cb["value"])
        last = cb
        if it == 0 and cb["seconds_setup"] + cb["seconds_per_call"] + 4 * cb["seconds_per_row"] > 60:
            # one sample already takes a minute: do not repeat it warmup+steps times
            vals = [cb["value"]]
            break
    value = float(np.mean(vals))
    npair_rows = npair * v * nrhs
    line = {"impl": "reference", "metric": "sigma_matvec_fp64_tflops", "value": value, "unit": "TFLOP/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": (kfix + 1) * flops_sigma / (value * 1e12) * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_string(cfg, c, nrhs, kfix, 0), "l2": "working set >> 126 MB L2"},
            "cpu_baseline": {"value": value, "unit": "TFLOP/s", "cores": last["cores"], "kind": "oracle", "sample": last["sample"]},
            "e2e": {"value": value, "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "note": f"extrapolated from sampled rows ({npair_rows} outputs per application; factor {last['extrapolation_factor']:.3g})"}
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------------------
def converged_solves(g, gi, torch, stream):
    """(p,omega) solves per second from CONVERGED batched GMRES solves (gfcc_solve_ip to the config's own tolerance, compaction and
    refill on): config 0 inside its own omega window (4 p x 8 omega, tol 1e-10) and config 1 at omega above the poles, where the
    paper's unpreconditioned GMRES converges on the synthetic spectrum (reading 23; 16 p x 2 omega, tol 1e-8)."""
    out = {}
    for name, cfg, ws, m in (("config0", 0, None, 400), ("config1", 1, [0.4, 0.5], 700)):
        c = gi.CONFIGS[cfg]
        s = gi.make_config(cfg, "cuda")
        h = g.gfcc_create(c["o"], c["v"], c["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"])
        g.gfcc_set_stream(h, stream)
        g.gfcc_set_option(h, "gmres_m", m)
        g.gfcc_set_option(h, "gmres_maxit", 4 * m)
        omegas = np.linspace(c["wlo"], c["whi"], c["nw"]) if ws is None else np.array(ws)
        targets = gi.targets(cfg)
        res = {}
        for label, comp in (("lockstep", -1.0), ("compaction", 0.125)):
            g.gfcc_set_option(h, "compact", comp)
            g.gfcc_solve_ip(h, targets, omegas, c["eta"], c["tol"], allow_noconv=True)          # warm-up (allocations)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(stream):
                e0.record(stream)
                g.gfcc_solve_ip(h, targets, omegas, c["eta"], c["tol"], allow_noconv=True)
                e1.record(stream)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            n = len(targets) * len(omegas)
            rel, its = g.gfcc_get_residuals(h, n)
            res[label] = {"ms": ms, "solves_per_s": n / (ms * 1e-3), "n_unconverged": int(g.gfcc_get_stat(h, "n_unconverged")),
                          "iterations_min_max": [int(its.min()), int(its.max())], "compactions": int(g.gfcc_get_stat(h, "compactions")),
                          "col_steps": g.gfcc_get_stat(h, "active_col_steps"), "lockstep_col_steps": g.gfcc_get_stat(h, "lockstep_col_steps")}
        best = max(res.values(), key=lambda r: r["solves_per_s"])
        out[name] = {"solves": len(targets) * len(omegas), "omega": [float(omegas[0]), float(omegas[-1])], "tol": c["tol"], "gmres_m": m,
                     "solves_per_s": best["solves_per_s"], **res}
        g.gfcc_destroy(h)
        del s
        torch.cuda.empty_cache()
    return out


# ---------------------------------------------------------------------------------------------------------
def main():
    args = parse()
    if args.cpu_baseline_only:
        return run_cpu_baseline_child(args)
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import gfcc_inputs as gi
    import paper_2010_04768_b200 as g
    from paper_2010_04768_b200 import sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    cfg = args.config
    c = gi.CONFIGS[cfg]
    o, v, Q = c["o"], c["v"], c["Q"]
    nrhs = c["np"] * c["nw"]
    kfix = args.kfix or KFIX[cfg]

    # ---- CPU baseline: started first; overlaps only input generation / gfcc_create / warm-up (rank 0, N = 1 only) ----
    cpu_child = None
    if world == 1 and not args.no_cpu_baseline and not args.cpu_baseline_serial:
        cpu_child = start_cpu_baseline_child(cfg)

    # ---- inputs (seeded, generated directly in HBM) and one-time intermediates ----
    t0 = time.time()
    s = gi.make_config(cfg, "cuda")
    torch.cuda.synchronize()
    t_inputs = time.time() - t0
    t0 = time.time()
    h = g.gfcc_create(o, v, Q, s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"])
    torch.cuda.synchronize()
    create_s = time.time() - t0
    flops_create = g.gfcc_get_stat(h, "flops_create")
    del s["Lchol"]
    torch.cuda.empty_cache()
    stream = torch.cuda.Stream()
    g.gfcc_set_stream(h, stream)
    g.gfcc_set_option(h, "gmres_fixed", kfix)
    g.gfcc_set_option(h, "max_batch", nrhs)
    if args.overlap >= 0:
        g.gfcc_set_option(h, "overlap", args.overlap)
    if args.panel_bytes > 0:
        g.gfcc_set_option(h, "panel_bytes", args.panel_bytes)
    if args.engine == "ozaki":
        g.gfcc_set_option(h, "ozaki_slices", args.slices)
        g.gfcc_set_option(h, "engine", 1)
        g.gfcc_set_option(h, "panel_bytes", 4.2e9)

    # rank r solves its own slice of the omega sweep (independent (p,omega) tasks; weak scaling)
    omegas = sharding.weak_scaling_grid(c["wlo"], c["whi"], c["nw"], max(world, 1), rank)
    targets = gi.targets(cfg)

    def step():
        return g.gfcc_solve_ip(h, targets, omegas, c["eta"], c["tol"])

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    flops_sigma = g.gfcc_get_stat(h, "flops_sigma")
    # roofline denominator measured IN THIS RUN: DMMA issue-rate probe on the same GPU, same stream, just before the timed region
    peak_in_run = g.gfcc_probe_fp64_peak(20000, 3, stream)
    cpu_result = None
    if cpu_child is not None:                       # the oracle sample must be over before the timed region starts
        cpu_result = finish_cpu_baseline_child(cpu_child, flops_sigma)
        cpu_child = None
    g.gfcc_get_stat(h, "reset_counters")
    overlap_on = args.overlap == 1
    if not overlap_on:      # per-launch events serialise the side streams, so with overlap the GEMM profile is a separate step
        g.gfcc_set_option(h, "profile_gemm", 1)
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        e0.record(stream)
        for _ in range(args.steps):
            G = step()
        e1.record(stream)
    barrier()
    sampler.stop_flag = True
    ms_total = e0.elapsed_time(e1)
    launches = g.gfcc_get_stat(h, "kernel_launches")
    napply = g.gfcc_get_stat(h, "sigma_applications")
    ms_prof = ms_total
    if overlap_on:
        g.gfcc_set_option(h, "profile_gemm", 1)
        with torch.cuda.stream(stream):
            e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e2.record(stream)
            step()
            e3.record(stream)
        barrier()
        ms_prof = e2.elapsed_time(e3)
    gemm_ms = g.gfcc_get_stat(h, "gemm_time_ms")
    gemm_flops = g.gfcc_get_stat(h, "gemm_flops_timed")
    gemm_n = g.gfcc_get_stat(h, "gemm_launches_timed")
    oz_ms, oz_ops, oz_fl, oz_n = (g.gfcc_get_stat(h, k) for k in ("oz_time_ms", "oz_ops_timed", "oz_flops_timed", "oz_launches_timed"))
    g.gfcc_set_option(h, "profile_gemm", 0)
    ms_total = sharding.max_over_ranks(ms_total, world, dist, "cuda")
    ms_step = ms_total / args.steps
    apps_per_step = napply / args.steps
    value = world * apps_per_step * flops_sigma / (ms_step * 1e-3) / 1e12
    rhs_steps_per_s = world * nrhs * kfix / (ms_step * 1e-3)

    line = {
        "metric": "sigma_matvec_fp64_tflops", "value": value, "unit": "TFLOP/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_string(cfg, c, nrhs, kfix, rank), "l2": "inputs and working set >> 126 MB L2 (no flush needed)",
                   "flop_model": "executed Cholesky-route model, SURVEY.md 8(d): real x complex = 2 real products, pair-packed o^4 term",
                   "flops_per_sigma_application": flops_sigma, "sigma_applications_per_step": apps_per_step,
                   "gmres_fixed_steps": kfix, "gmres_m_memory_limit": g.gfcc_get_stat(h, "gmres_m_memory_limit"),
                   "gmres_m_note": "gmres_m_memory_limit = longest Krylov basis (batch vectors) the free device memory allows beside the "
                                   "resident intermediates at this batch width; the timed step runs gmres_fixed_steps Arnoldi steps",
                   "overlap": int(overlap_on),
                   "gemm_engine": ("dgemm_ws_kernel (FP64 DMMA, warp-specialised)" if args.engine == "dmma" else
                                   f"ozaki_int8 x{args.slices} slices for S6, S8-S11 (tcgen05.mma kind::i8, exact int32 accumulation, FP64-accurate; "
                                   "NOT the graded FP64 DMMA engine), rest on the DMMA engine"),
                   "panel_ni": g.gfcc_get_stat(h, "panel_ni")},
        "rhs_arnoldi_steps_per_s": rhs_steps_per_s,
        "rhs_arnoldi_steps_note": "(right-hand sides x Arnoldi steps) per second in the fixed-step timing mode; NOT a solve rate -- "
                                  "converged (p,omega) solves per second are in `solves`",
        "pct_fp64_peak_measured": 100.0 * value / world / peak_in_run,
        "create_s": create_s, "create_tflops": flops_create / create_s / 1e12, "inputs_s": t_inputs,
        "device_bytes": g.gfcc_get_stat(h, "bytes_device"), "gpu_launches": int(launches),
    }
    line["clocks"] = sampler.summary()

    # ---- roofline of the dominant kernel (dgemm_dmma_kernel): CUDA events around every launch, on the launching stream ----
    mp = measured_peaks()
    achieved = gemm_flops / (gemm_ms * 1e-3) / 1e12 if gemm_ms > 0 else 0.0
    line["roofline"] = {
        "kernel": "gfcc::dgemm_ws_kernel (all GEMM-engine launches of the timed region)",
        "bound": "tensor", "achieved": achieved, "peak": peak_in_run, "unit": "TFLOP/s", "frac": achieved / peak_in_run,
        "peak_source": "FP64 DMMA.8x8x4 issue-rate ceiling measured IN THIS RUN by gfcc_probe_fp64_peak (register-only DMMA loop on every SM, "
                       "CUDA events, right before the timed region); MEASURED_PEAKS.json has no FP64 entry",
        "peak_round1_constant": FP64_DMMA_PEAK_R1,
        "peak_alt_bf16_ratio": (mp["bf16_tflops_sustained"] * 40.0 / 2250.0) if mp else None,
        "peak_alt_note": "sustained bf16 peak of MEASURED_PEAKS.json x nominal FP64:bf16 ratio 40/2250 (fallback rule; lower than the "
                         "directly measured DMMA ceiling, so the stricter denominator is used for frac)",
        "launches": int(gemm_n), "avg_launch_ms": gemm_ms / max(gemm_n, 1), "share_of_step": gemm_ms / ms_prof if ms_prof > 0 else None,
        "algorithmic_flops": gemm_flops,
    }
    tr = ncu_traffic(cfg)
    line["roofline"]["traffic"] = tr["bytes"] if tr else None
    line["roofline"]["traffic_note"] = (
        f"dram__bytes_read.sum + dram__bytes_write.sum of ONE launch from ncu --set full, read from {tr['source']}: launch '{tr['launch']}', "
        f"{tr['shape']}, the most frequent big launch of this step; its algorithmic bytes (A + B + C once) are {tr['algorithmic_bytes']:.3g}"
        if tr else "no ncu capture of this config's launch shapes in profiles/r2_gemm_ncu_traffic.csv")

    if args.engine == "ozaki" and oz_ms > 0:
        i8_peak = (mp["bf16_tflops_sustained"] * 2.0) if mp else 2.0 * 1365.7
        r = line["roofline"]
        line["roofline_dmma_part"] = {k: r[k] for k in ("achieved", "launches", "share_of_step")}
        line["roofline"] = {
            "kernel": "gfcc::oz_igemm_kernel (INT8 tcgen05 launches of the timed region: S6, S8-S11)", "bound": "tensor",
            "achieved": oz_ops / (oz_ms * 1e-3) / 1e12, "peak": i8_peak, "unit": "TFLOP/s", "frac": oz_ops / (oz_ms * 1e-3) / 1e12 / i8_peak,
            "peak_source": "int8 dense = sustained bf16 of MEASURED_PEAKS.json x nominal ratio 4.5/2.25 (no measured int8 entry); unit is int8 TOP/s",
            "peak_alt_burst": (mp["bf16_tflops"] * 2.0) if mp else None,
            "launches": int(oz_n), "avg_launch_ms": oz_ms / max(oz_n, 1), "share_of_step": oz_ms / ms_prof if ms_prof > 0 else None,
            "algorithmic_flops": oz_fl, "fp64_equivalent_tflops": oz_fl / (oz_ms * 1e-3) / 1e12,
            "int8_ops": oz_ops, "traffic": None,
            "note": "int8 ops = 2MNK x S(S+1)/2 digit-matrix products; fp64_equivalent = 2MNK / time"}
        line["pct_fp64_peak_note"] = "above 100 % by construction: the work runs on the INT8 pipe, FP64 DMMA peak is only the yardstick"

    # ---- end to end through the C ABI with HOST buffers: one batched sigma application, copies inside the call ----
    if not args.no_e2e and rank == 0:
        try:
            X1, X2 = gi.trial_vectors(o, v, nrhs, gi.seed_of(cfg), "cuda")
            X1h = torch.empty(X1.shape, dtype=X1.dtype, pin_memory=True).copy_(X1)
            X2h = torch.empty(X2.shape, dtype=X2.dtype, pin_memory=True).copy_(X2)
            del X1, X2
            torch.cuda.empty_cache()
            wr = np.repeat(omegas, c["np"])[:nrhs] if len(omegas) * c["np"] >= nrhs else np.resize(omegas, nrhs)
            S1p = torch.empty(X1h.shape, dtype=X1h.dtype, pin_memory=True)
            S2p = torch.empty(X2h.shape, dtype=X2h.dtype, pin_memory=True)
            g.gfcc_sigma_ip_host(h, wr, c["eta"], X1h.numpy(), X2h.numpy(), out=(S1p, S2p))   # warm-up
            nrep = 2 if cfg >= 3 else 3
            t0 = time.perf_counter()
            for _ in range(nrep):
                S1h, S2h = g.gfcc_sigma_ip_host(h, wr, c["eta"], X1h.numpy(), X2h.numpy(), out=(S1p, S2p))
            dt = (time.perf_counter() - t0) / nrep
            nb = X1h.numel() * 16 + X2h.numel() * 16
            line["e2e"] = {"value": flops_sigma / dt / 1e12, "unit": "TFLOP/s", "h2d_bytes_per_step": int(nb + 8 * nrhs),
                           "d2h_bytes_per_step": int(nb), "ms_per_step": dt * 1e3,
                           "what": "gfcc_sigma_ip_host: X1,X2 from pinned host memory, S1,S2 back to pinned host memory, copies inside the timed call",
                           "note": "the timed STEP itself (gfcc_solve_ip) already takes host arrays p[], omega[] and returns G on the host; its only "
                                   "device-resident input is the handle built by gfcc_create, so `value` is end to end for the solve step and this "
                                   "entry adds the sigma call whose vectors (5.5 GB each way at config 4) cross PCIe"}
        except Exception as ex:   # noqa: BLE001
            line["e2e"] = {"value": None, "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0, "error": str(ex)[:200]}
    # ---- extra (not the headline): the same step on the INT8 tensor-core engine, 1 warm-up + 1 timed step ----
    if args.engine == "dmma" and not args.no_ozaki_extra and cfg >= 1:
        try:
            g.gfcc_set_option(h, "ozaki_slices", args.slices)
            g.gfcc_set_option(h, "engine", 1)
            g.gfcc_set_option(h, "panel_bytes", 4.2e9)
            step()
            g.gfcc_set_option(h, "profile_gemm", 1)
            barrier()
            with torch.cuda.stream(stream):
                e4, e5 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e4.record(stream)
                step()
                e5.record(stream)
            barrier()
            ms_oz = sharding.max_over_ranks(e4.elapsed_time(e5), world, dist, "cuda")
            o_ms, o_ops, o_fl = (g.gfcc_get_stat(h, k) for k in ("oz_time_ms", "oz_ops_timed", "oz_flops_timed"))
            g.gfcc_set_option(h, "profile_gemm", 0)
            line["ozaki_int8"] = {
                "value": world * apps_per_step * flops_sigma / (ms_oz * 1e-3) / 1e12, "unit": "TFLOP/s (FP64-equivalent, same flop model)",
                "ms_per_step": ms_oz, "slices": args.slices, "speedup_vs_dmma_step": ms_step / ms_oz,
                "int8_tops_in_kernel": o_ops / (o_ms * 1e-3) / 1e12 if o_ms > 0 else None,
                "fp64_equivalent_tflops_in_kernel": o_fl / (o_ms * 1e-3) / 1e12 if o_ms > 0 else None,
                "kernel_share_of_step": o_ms / ms_oz if ms_oz > 0 else None, "oz_fail": g.gfcc_get_stat(h, "oz_fail"),
                "note": "S6, S8-S11 on tcgen05.mma kind::i8 with error-free slicing (FP64-accurate: sigma parity 1e-10 in tests/test_gpu_ozaki.py); "
                        "reported beside, not instead of, the graded FP64 DMMA number"}
        except Exception as ex:   # noqa: BLE001
            line["ozaki_int8"] = {"value": None, "error": str(ex)[:200]}
    g.gfcc_destroy(h)
    del s
    torch.cuda.empty_cache()

    # ---- converged (p,omega) solves per second: real batched solves to the config's tolerance (rank 0, N = 1) ----
    if world == 1 and not args.no_solves:
        try:
            line["solves"] = converged_solves(g, gi, torch, stream)
            line["solves_per_s"] = line["solves"]["config0"]["solves_per_s"]
        except Exception as ex:   # noqa: BLE001
            line["solves"] = {"error": str(ex)[:200]}

    # ---- CPU baseline: the oracle on the host cores, bounded sample (rank 0, N = 1 only) ----
    if cpu_result is not None:
        line["cpu_baseline"] = cpu_result
    elif world == 1 and not args.no_cpu_baseline:
        try:
            cb = cpu_baseline(cfg, c, nrhs, flops_sigma)
            cb.pop("seconds_full", None)
            line["cpu_baseline"] = cb
        except Exception as ex:   # noqa: BLE001
            line["cpu_baseline"] = {"value": None, "unit": "TFLOP/s", "cores": None, "kind": "oracle", "sample": f"failed: {str(ex)[:200]}"}
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
