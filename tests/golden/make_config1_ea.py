#!/usr/bin/env python
"""Writes tests/golden/config1_ea.npz: values of the oracle's DEFINITION-FORM EA / advanced part (oracle/gfcc_oracle.cpp
build_ea, sigma_ea_one, orc_bra_ea, orc_gmres_ea; Eq. 6, second terms of Eq. 7-8) at the full size of BASELINE.json
config 1 (o=40, v=160, Q=600), where its O(v^4) arrays (2 x 5.2 GB) take the better part of an hour to build.

    python tests/golden/make_config1_ea.py [--out tests/golden/config1_ea.npz] [--kfix 8]

Imports ONLY `oracle/` and `gfcc_inputs/`; runs on the host cores (inputs drawn on the CPU: the GPU test uses the same bits).
Stored: sigma_EA of two seeded trial vectors (gfcc_inputs.trial_vectors_ea) at sampled rows, c_p . Y for three p, and for the
target q = o (lowest virtual) at omega = -0.4 (inside config 1's window) the oracle GMRES residual history of `kfix` steps,
the unique kfix-step iterate at sampled rows and G^A_pq from it.
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import gfcc_inputs as gi  # noqa: E402
import oracle  # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_ea.npz"))
    ap.add_argument("--kfix", type=int, default=8)
    ap.add_argument("--config", type=int, default=1)
    args = ap.parse_args()
    cfg = args.config
    c = gi.CONFIGS[cfg]
    o, v, Q = c["o"], c["v"], c["Q"]
    s = gi.make_config(cfg, "cpu")
    host = {k: s[k].numpy() for k in ("fock", "T1", "T2p", "L1", "L2p", "Lchol")}
    nsel = 2
    Y1, Y2 = gi.trial_vectors_ea(o, v, nsel, gi.seed_of(cfg), "cpu")
    Y1h, Y2h = Y1.numpy(), Y2.numpy()
    w = np.array([c["wlo"], c["whi"]])
    rng = np.random.default_rng(300 + cfg)
    rows = [(0, 0, 1), (o - 1, v - 2, v - 1), (o // 2, 1, v // 2), (1, 0, v - 1)]
    while len(rows) < 10:
        a, b = sorted(rng.choice(v, 2, replace=False))
        rows.append((int(rng.integers(0, o)), int(a), int(b)))
    rows = np.array(rows, dtype=np.int32)
    s1rows = np.array([0, v // 3, v - 1], dtype=np.int32)
    t0 = time.time()
    orc = oracle.Oracle(o, v, Q, host["fock"], host["T1"], host["T2p"], host["L1"], host["L2p"], host["Lchol"],
                        oracle.MODE_DEF | oracle.MODE_EA)
    t_build = time.time() - t0
    print(f"definition-form IP + EA intermediates: {t_build:.1f} s", flush=True)
    t0 = time.time()
    S1, S2 = orc.sigma_ea(w, c["eta"], Y1h, Y2h)
    t_sigma = (time.time() - t0) / nsel
    print(f"sigma_EA: {t_sigma:.1f} s per RHS", flush=True)
    S1s = S1[:, s1rows].T.copy()
    S2s = np.stack([S2[:, j, a, b] for (j, a, b) in rows], axis=0)
    plist = np.array([o, o + 5, o - 1], dtype=np.int32)
    GA = np.empty((nsel, len(plist)), dtype=np.complex128)
    for ip, p in enumerate(plist):
        c1, c2 = orc.bra_ea(int(p))
        for r in range(nsel):
            GA[r, ip] = orc.bra_dot_ea(c1, c2, Y1h[r], Y2h[r])
    q, om = o, -0.4
    t0 = time.time()
    y1, y2, nit, rr, hist = orc.gmres_ea(q, om, c["eta"], 1e-30, m=args.kfix, maxit=args.kfix + 1, x0kind=1, history=True)
    print(f"GMRES {nit} applications in {time.time() - t0:.1f} s, relres {rr:.3e}", flush=True)
    Gk = np.array([orc.bra_dot_ea(*orc.bra_ea(int(p)), y1, y2) for p in plist])
    np.savez(args.out, cfg=cfg, nsel=nsel, omega=w, eta=c["eta"], rows=rows, s1rows=s1rows, S1s=S1s, S2s=S2s, plist=plist, GA=GA,
             q=q, om=om, kfix=args.kfix, hist=hist, Y1k=y1, Y2k=np.array([y2[j, a, b] for (j, a, b) in rows]), Gk=Gk,
             scale2=np.abs(S2).max(), scale1=np.abs(S1).max(), timing=np.array([t_build, t_sigma]), threads=oracle.threads())
    print("wrote", args.out, flush=True)


if __name__ == "__main__":
    main()
