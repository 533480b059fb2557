"""Measurement tool (not product): micro-benchmarks of the building blocks (B200): FP64 DMMA ceiling, the GEMM engine on square and on the sigma-shaped
problems of a config, HBM copy.  Used for the roofline notes in DESIGN.md / profiles/ and as the short command ncu wraps.

    python bench_micro.py [--probe] [--square N] [--sigma-shapes CFG] [--ozaki-shapes CFG] [--slices S] [--reps R]
"""
import argparse
import json
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

import torch

import paper_2010_04768_b200 as g

SHAPES = {   # (o, v, Q, nrhs)
    1: (40, 160, 600, 64), 2: (80, 320, 1200, 64), 3: (120, 480, 1800, 32), 4: (180, 660, 2500, 16),
}


def time_gemm(M, N, K, ta=False, tb=False, reps=3):
    A = torch.randn((K, M) if ta else (M, K), dtype=torch.float64, device="cuda")
    B = torch.randn((N, K) if tb else (K, N), dtype=torch.float64, device="cuda")
    C = torch.empty((M, N), dtype=torch.float64, device="cuda")
    Av, Bv = (A.t() if ta else A), (B.t() if tb else B)
    g.gfcc_dgemm(Av, Bv, C)
    torch.cuda.synchronize()
    best = 1e30
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g.gfcc_dgemm(Av, Bv, C)
        e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    return {"M": M, "N": N, "K": K, "ta": ta, "tb": tb, "ms": best, "tflops": 2.0 * M * N * K / best / 1e9}


def time_ozaki(M, N, K, ta=False, S=7, reps=2):
    """gfcc_dgemm_ozaki (INT8 tensor-core engine): CUDA-event times of the slicing passes and of the tcgen05 kernel"""
    A = torch.randn((K, M) if ta else (M, K), dtype=torch.float64, device="cuda")
    B = torch.randn((K, N), dtype=torch.float64, device="cuda")
    C = torch.zeros((M, N), dtype=torch.float64, device="cuda")
    Av = A.t() if ta else A
    best = (1e30, 1e30)
    for _ in range(reps):
        _, ms_s, ms_g = g.gfcc_dgemm_ozaki(Av, B, C, nslices=S, return_times=True)
        best = min(best, (ms_g, ms_s))
    ms_g, ms_s = best
    return {"M": M, "N": N, "K": K, "ta": ta, "slices": S, "ms_gemm": ms_g, "ms_slice": ms_s,
            "fp64_equiv_tflops": 2.0 * M * N * K / ms_g / 1e9, "int8_tops": 2.0 * M * N * K * (S * (S + 1) // 2) / ms_g / 1e9}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--probe", action="store_true")
    ap.add_argument("--square", type=int, default=0)
    ap.add_argument("--sigma-shapes", type=int, default=0)
    ap.add_argument("--ozaki-shapes", type=int, default=0)
    ap.add_argument("--slices", type=int, default=7)
    ap.add_argument("--reps", type=int, default=3)
    ap.add_argument("--sigma-once", type=int, default=-1,
                    help="config id: gfcc_create + ONE batched gfcc_sigma_ip on the seeded trial vectors (the short command ncu wraps "
                         "with NVTX range filters, e.g. --nvtx --nvtx-include 'S11 Z4 = T2 V/')")
    ap.add_argument("--mor", type=int, default=-1,
                    help="config id: MOR step at a size that means something (SURVEY 8f rows 1, 3): two levels of converged solves at "
                         "omega above the poles, Gram-Schmidt + projection, reduced solves on a fine grid; times per phase and the "
                         "interpolation error against direct solves")
    ap.add_argument("--adaptive", type=int, default=-1,
                    help="config id: gfcc_spectral_adaptive (Alg. 1 level loop) over a window above the poles; wall time, levels, m, "
                         "and A at the sampled points against direct converged solves")
    ap.add_argument("--ea-once", type=int, default=-1,
                    help="config id (0 or 1): gfcc_create + EA preparation + timed batched gfcc_sigma_ea applications on seeded trial vectors")
    a = ap.parse_args()
    out = {}
    if a.ea_once >= 0:
        import gfcc_inputs as gi
        c = gi.CONFIGS[a.ea_once]
        s = gi.make_config(a.ea_once, "cuda")
        h = g.gfcc_create(c["o"], c["v"], c["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"])
        nrhs = 32
        Y1, Y2 = gi.trial_vectors_ea(c["o"], c["v"], nrhs, gi.seed_of(a.ea_once), "cuda")
        w = [0.3] * nrhs
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g.gfcc_sigma_ea(h, w, c["eta"], Y1, Y2)          # first call: builds W_abej and the workspace
        e1.record()
        torch.cuda.synchronize()
        first_ms = e0.elapsed_time(e1)
        best, fl = 1e30, 0.0
        for _ in range(max(1, a.reps)):
            f0 = g.gfcc_get_stat(h, "flops_executed")
            e0.record()
            g.gfcc_sigma_ea(h, w, c["eta"], Y1, Y2)
            e1.record()
            torch.cuda.synchronize()
            fl = g.gfcc_get_stat(h, "flops_executed") - f0
            best = min(best, e0.elapsed_time(e1))
        out["ea_once"] = {"config": a.ea_once, "nrhs": nrhs, "first_call_ms (incl. W_abej build)": first_ms, "ms": best,
                          "executed_gemm_flops": fl, "tflops_executed": fl / best / 1e9}
        g.gfcc_destroy(h)
    if a.adaptive >= 0:
        import time
        import numpy as np
        import gfcc_inputs as gi
        c = gi.CONFIGS[a.adaptive]
        s = gi.make_config(a.adaptive, "cuda")
        h = g.gfcc_create(c["o"], c["v"], c["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"])
        targets = gi.targets(a.adaptive)[:4]
        wmin, wmax, dw, eta, tol = 0.40, 0.56, 0.01, c["eta"], 1e-8
        g.gfcc_set_option(h, "gmres_m", 700)
        g.gfcc_set_option(h, "gmres_maxit", 2800)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        r = g.gfcc_spectral_adaptive(h, targets, wmin, wmax, dw, eta, tol, spec_tol=1e-3, droptol=1e-8)
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        lev = r["level_of"]
        sampled = [int(k) for k in np.nonzero(lev)[0]]
        chk = [sampled[1], sampled[len(sampled) // 2]]
        Gd = g.gfcc_solve_ip(h, targets, [float(r["w"][k]) for k in chk], eta, tol)
        Ad = [float(np.trace(Gd[q]).imag / np.pi) for q in range(len(chk))]
        out["adaptive"] = {"config": a.adaptive, "targets": targets, "window": [wmin, wmax, dw], "levels": int(r["levels"]), "m": int(r["m"]),
                           "points_per_level": [int((lev == L).sum()) for L in range(1, int(r["levels"]) + 1)], "wall_s": wall,
                           "sampled_omega": [float(r["w"][k]) for k in sampled], "check_omega": [float(r["w"][k]) for k in chk],
                           "A_model": [float(r["A"][k]) for k in chk], "A_direct": Ad,
                           "rel_err": [abs(float(r["A"][k]) - Ad[q]) / abs(Ad[q]) for q, k in enumerate(chk)],
                           "A_fine": [float(x) for x in r["A"]]}
        g.gfcc_destroy(h)
    if a.mor >= 0:
        import numpy as np
        import gfcc_inputs as gi
        c = gi.CONFIGS[a.mor]
        s = gi.make_config(a.mor, "cuda")
        h = g.gfcc_create(c["o"], c["v"], c["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"])
        targets = gi.targets(a.mor)[:4]
        wmin, wmax, dw, eta, tol = 0.40, 0.56, 0.01, c["eta"], 1e-8
        fine = wmin + dw * np.arange(int(round((wmax - wmin) / dw)) + 1)
        g.gfcc_set_option(h, "gmres_m", 700)
        g.gfcc_set_option(h, "gmres_maxit", 2800)
        g.gfcc_mor_reset(h, 2 * len(targets) * 9)

        def timed(fn):
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            r = fn()
            e1.record()
            torch.cuda.synchronize()
            return r, e0.elapsed_time(e1)

        levels = [[fine[0], fine[len(fine) // 2], fine[-1]], [fine[len(fine) // 4], fine[3 * len(fine) // 4]]]
        rec = []
        for lv, ws in enumerate(levels):
            (G, X1, X2), ms_solve = timed(lambda: g.gfcc_solve_ip(h, targets, ws, eta, tol, return_x=True))
            its = g.gfcc_get_residuals(h, len(targets) * len(ws))[1]
            m, ms_ext = timed(lambda: g.gfcc_mor_extend(h, X1, X2, 1e-8))
            del X1, X2
            (Gh, A), ms_red = timed(lambda: g.gfcc_mor_solve(h, targets, fine, eta))
            rec.append({"level": lv + 1, "omegas": [float(w) for w in ws], "m": m, "solve_ms": ms_solve, "gmres_iterations_min_max": [int(its.min()), int(its.max())],
                        "extend_ms (Gram-Schmidt + projection)": ms_ext, "reduced_solves_ms (fine grid, %d points)" % len(fine): ms_red,
                        "A_fine": [float(x) for x in A]})
        # interpolation check at grid points that were NOT sampled: direct converged solves
        chk = [fine[1], fine[len(fine) // 2 + 2]]
        Gd = g.gfcc_solve_ip(h, targets, chk, eta, tol)
        Ad = [float(np.trace(Gd[k]).imag / np.pi) for k in range(len(chk))]
        idx = [1, len(fine) // 2 + 2]
        out["mor"] = {"config": a.mor, "targets": targets, "window": [wmin, wmax, dw], "levels": rec,
                      "check_omegas": [float(w) for w in chk], "A_direct": Ad, "A_model": [rec[-1]["A_fine"][k] for k in idx],
                      "rel_err": [abs(rec[-1]["A_fine"][k] - Ad[q]) / abs(Ad[q]) for q, k in enumerate(idx)]}
        g.gfcc_destroy(h)
    if a.sigma_once >= 0:
        import gfcc_inputs as gi
        c = gi.CONFIGS[a.sigma_once]
        s = gi.make_config(a.sigma_once, "cuda")
        h = g.gfcc_create(c["o"], c["v"], c["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"])
        del s["Lchol"]
        torch.cuda.empty_cache()
        nrhs = c["np"] * c["nw"] if a.sigma_once >= 2 else 64
        X1, X2 = gi.trial_vectors(c["o"], c["v"], nrhs, gi.seed_of(a.sigma_once), "cuda")
        w = [c["wlo"]] * nrhs
        for _ in range(max(1, a.reps if a.reps < 3 else 1)):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            g.gfcc_sigma_ip(h, w, c["eta"], X1, X2)
            e1.record()
            torch.cuda.synchronize()
        out["sigma_once"] = {"config": a.sigma_once, "nrhs": nrhs, "ms": e0.elapsed_time(e1), "panel_ni": g.gfcc_get_stat(h, "panel_ni"),
                             "tflops": g.gfcc_get_stat(h, "flops_sigma") / e0.elapsed_time(e1) / 1e9}
        g.gfcc_destroy(h)
    if a.probe:
        out["fp64_dmma_peak_tflops"] = g.gfcc_probe_fp64_peak(20000, 5)
        x = torch.empty(1 << 28, dtype=torch.float64, device="cuda")
        y = torch.empty_like(x)
        y.copy_(x)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        y.copy_(x)
        e1.record()
        torch.cuda.synchronize()
        out["hbm_copy_gbs"] = 2 * x.numel() * 8 / e0.elapsed_time(e1) / 1e6
        del x, y
    if a.square:
        n = a.square
        out["square"] = [time_gemm(n, n, n, ta, tb, a.reps) for ta in (False, True) for tb in (False, True)]
    if a.sigma_shapes:
        o, v, Q, nrhs = SHAPES[a.sigma_shapes]
        ov, ld, Nc = o * v, o * 2 * nrhs, 2 * nrhs
        ni = max(1, min(o, int(3.2e9 // (ov * 8 * v))))
        shapes = [("S1  Y = Lov XU", Q, ld, ov, False, False), ("S7  Z = Lm^T Y", ov, ld, Q, True, False),
                  ("S8  K2 panel build", ni * o, v * v, Q, True, False), ("S9  Z -= K2 XU (panel)", ni * v, ld, ov, False, False),
                  ("S6  W_mnij x2", o * (o - 1) // 2, v * Nc, o * (o - 1) // 2, False, False)]
        out["sigma_shapes"] = []
        for name, M, N, K, ta, tb in shapes:
            r = time_gemm(M, N, K, ta, tb, a.reps)
            r["name"] = name
            out["sigma_shapes"].append(r)
    if a.ozaki_shapes:
        o, v, Q, nrhs = SHAPES[a.ozaki_shapes]
        ov, ld = o * v, o * 2 * nrhs
        ni = max(1, min(o, int(4.2e9 // (ov * 8 * v))))
        shapes = [("S8  K2 panel build (short K: register-accumulating kernel)", ni * o, v * v, Q, True),
                  ("S10 K4 panel build (short K)", ov, ni * v, Q, True),
                  ("S9  Z -= K2 XU (panel; long K: 128 x 256 kernel)", ni * v, ld, ov, False)]
        out["ozaki_shapes"] = []
        for name, M, N, K, ta in shapes:
            r = time_ozaki(M, N, K, ta, a.slices, max(1, min(a.reps, 2)))
            r["name"] = name
            out["ozaki_shapes"].append(r)
    print(json.dumps(out))


if __name__ == "__main__":
    main()
