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
    a = ap.parse_args()
    out = {}
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
