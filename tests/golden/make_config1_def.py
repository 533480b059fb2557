#!/usr/bin/env python
"""Writes tests/golden/config1_def.npz: values of the DEFINITION-FORM oracle (oracle/gfcc_oracle.cpp build_def,
sigma_def_one, orc_gmres_hist: explicit <pq||rs> blocks, plain loops) at the full size of BASELINE.json config 1
(o=40, v=160, Q=600), where building it takes minutes (1.3 GB <ov||vv> block) -- too long for the test suites.

    python tests/golden/make_config1_def.py [--out tests/golden/config1_def.npz] [--steps 80]

Imports ONLY `oracle/` and `gfcc_inputs/`; runs on the host cores.  Stored:
  S1def [n1, 2], S2def [ntrip, 2]  definition-form sigma of the seeded trial vectors (RHS 0 and 63 of the 64-RHS batch) at the
                                   same rows tests/golden/make_rows.py samples -> pins the ROW-SAMPLED oracle (the only
                                   checker at configs 1-4) against the definition form at o = 40
  hist [nw, steps+1]               oracle GMRES (no restart, x0 = zeroth-order guess) relative-residual history for the
                                   target p = o-1 at omega = -0.25 (inside config 1's window) and +0.4 (above the poles):
                                   the oracle's verdict on DESIGN.md reading 23 (stagnation inside the window)
  X1k [nw, o], X2k [nw, ntrip]     the k-step iterate (k = 25; unique, reading 19) at sampled rows
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

import gfcc_inputs as gi  # noqa: E402
import oracle  # noqa: E402
from make_rows import triples  # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_def.npz"))
    ap.add_argument("--steps", type=int, default=80)
    ap.add_argument("--kfix", type=int, default=25)
    args = ap.parse_args()
    cfg = 1
    c = gi.CONFIGS[cfg]
    o, v, Q = c["o"], c["v"], c["Q"]
    s = gi.make_config(cfg, "cpu")
    host = {k: s[k].numpy() for k in ("fock", "T1", "T2p", "L1", "L2p", "Lchol")}
    nrhs = 64
    X1, X2 = gi.trial_vectors(o, v, nrhs, gi.seed_of(cfg), "cpu")
    rsel = [0, nrhs - 1]
    X1h, X2h = X1[rsel].numpy(), X2[rsel].numpy()
    w = np.resize(np.linspace(c["wlo"], c["whi"], c["nw"]), nrhs)
    trip = triples(o, v, 8, 100 + cfg)
    s1rows = np.array([0, o - 1], dtype=np.int32)
    t0 = time.time()
    orc = oracle.Oracle(o, v, Q, host["fock"], host["T1"], host["T2p"], host["L1"], host["L2p"], host["Lchol"], oracle.MODE_DEF)
    t_build = time.time() - t0
    print(f"definition-form intermediates: {t_build:.1f} s", flush=True)
    t0 = time.time()
    S1, S2 = orc.sigma(w[rsel], c["eta"], X1h, X2h)
    t_sigma = (time.time() - t0) / len(rsel)
    S1def = S1[:, s1rows].T.copy()
    S2def = np.stack([S2[:, i, j, a] for (i, j, a) in trip], axis=0)
    print(f"sigma: {t_sigma:.1f} s per RHS", flush=True)

    p = o - 1
    ws = np.array([-0.25, 0.4])
    hist = np.empty((len(ws), args.steps + 1))
    X1k = np.empty((len(ws), o), dtype=np.complex128)
    X2k = np.empty((len(ws), len(trip)), dtype=np.complex128)
    for iw, om in enumerate(ws):
        t0 = time.time()
        _, _, nit, rr, hh = orc.gmres(p, om, c["eta"], 1e-30, m=args.steps, maxit=args.steps + 1, x0kind=1, history=True)
        hist[iw] = hh
        x1, x2, nit2, rr2 = orc.gmres(p, om, c["eta"], 1e-30, m=args.kfix, maxit=args.kfix + 1, x0kind=1)
        X1k[iw] = x1
        X2k[iw] = np.array([x2[i, j, a] for (i, j, a) in trip])
        print(f"omega {om}: {nit} + {nit2} sigma applications in {time.time() - t0:.1f} s; relres after {args.steps} steps {rr:.3e}, "
              f"after {args.kfix} steps {rr2:.3e}", flush=True)
    np.savez(args.out, cfg=cfg, nrhs=nrhs, rsel=np.array(rsel, dtype=np.int32), omega=w, trip=trip, s1rows=s1rows, S1def=S1def,
             S2def=S2def, p=p, ws=ws, eta=c["eta"], hist=hist, kfix=args.kfix, X1k=X1k, X2k=X2k,
             timing=np.array([t_build, t_sigma]), threads=oracle.threads())
    print("wrote", args.out, flush=True)


if __name__ == "__main__":
    main()
