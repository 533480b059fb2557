"""Pins of the level-loop oracle (oracle/workflow.py; Alg. 1, Eq. 12-13) against what
the paper and the mathematics fix (run with -m "not gpu"):
  (m) the paper's worked example of Eq. 13: [-0.8, -0.4] a.u. with dw = 0.01 gives L_max <= 5 (tests/golden/eq13_example.txt);
  (n) Eq. 12 counts: 3 points at level 1, at most 2^(L-1) at level L > 1; never more than L_max levels; every sampled point is
      a point of the fine grid, sampled once, both ends included;
  (o) closed form T = Lambda = L = 0: the level-1 subspace already contains every b_p, so the model is exact, A(omega) is the
      sum of Lorentzians on the whole fine grid and the refinement stops by itself;
  (p) interpolation survives the level loop: at every sampled frequency the final G^ equals the UNREDUCED dense solve;
  (q) with spec_tol = 0 and enough levels every grid point is sampled and the model reproduces the dense spectral function
      on the whole grid (brute force).
"""
import os

import numpy as np

import oracle
from oracle import workflow
from gfcc_testutil import random_system

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "eq13_example.txt")


def _setup(o=4, v=5, Q=6, seed=31, **kw):
    s = random_system(o, v, Q, seed=seed, t_scale=0.05, l_scale=0.15, **kw)
    orc = oracle.Oracle(s["o"], s["v"], s["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"], oracle.MODE_DEF)
    H = orc.dense_hbar()
    plist = [o - 1, o - 2, o + 1]
    B = np.stack([orc.pack(*orc.rhs(p)).real for p in plist], axis=1)
    C = np.stack([orc.pack(*orc.bra(q)) for q in plist], axis=1)
    return s, orc, H, plist, B, C


def test_eq13_worked_example_from_the_paper():
    vals = dict(line.split("=") for line in open(GOLDEN).read().split() if "=" in line)
    wmin, wmax, dw = float(vals["wmin"]), float(vals["wmax"]), float(vals["dw"])
    assert workflow.level_bound(wmin, wmax, dw) == int(vals["Lmax"]) == 5
    assert len(workflow.fine_grid(wmin, wmax, dw)) == int(vals["Ntot"]) == 41
    # Eq. 12 / 13 consistency: sum of the per-level maxima up to L_max does not exceed N_tot
    assert 3 + sum(2 ** (L - 1) for L in range(2, 6)) <= 41


def test_eq12_counts_and_grid_membership():
    s, orc, H, plist, B, C = _setup()
    r = workflow.run(H, B, C, -1.2, -0.2, 0.01, 0.02, spec_tol=1e-6)
    lo = r["level_of"]
    assert len(r["w"]) == 101 and abs(r["w"][-1] + 0.2) < 1e-12
    assert lo[0] == 1 and lo[-1] == 1 and lo[50] == 1 and (lo == 1).sum() == 3
    assert 1 <= r["levels"] <= workflow.level_bound(-1.2, -0.2, 0.01) == 6
    for L in range(2, r["levels"] + 1):
        assert 1 <= (lo == L).sum() <= 2 ** (L - 1)
    assert (lo > r["levels"]).sum() == 0
    assert r["m"] <= 2 * len(plist) * int((lo > 0).sum())
    # max_levels caps the loop
    r2 = workflow.run(H, B, C, -1.2, -0.2, 0.01, 0.02, spec_tol=1e-6, max_levels=2)
    assert r2["levels"] == 2 and (r2["level_of"] > 0).sum() == 5


def test_closed_form_is_exact_after_level_one():
    o, v = 3, 4
    s = random_system(o, v, 2, seed=5, diag_f=True)
    for k in ("T1", "L1", "T2p", "L2p", "Lchol"):
        s[k] = np.zeros_like(s[k])
    orc = oracle.Oracle(o, v, 2, s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"], oracle.MODE_DEF)
    H = orc.dense_hbar()
    plist = [0, 1, 2]
    B = np.stack([orc.pack(*orc.rhs(p)).real for p in plist], axis=1)
    C = np.stack([orc.pack(*orc.bra(q)) for q in plist], axis=1)
    eta = 0.03
    r = workflow.run(H, B, C, -2.2, -0.8, 0.02, eta, spec_tol=1e-9)
    eps = np.diag(s["fock"])[:o]
    A_ref = sum(eta / ((r["w"] - e) ** 2 + eta ** 2) for e in eps) / np.pi
    assert np.abs(r["A"] - A_ref).max() < 1e-12 * A_ref.max()
    assert r["m"] == o                       # span{e_p}: imaginary parts and later samples are all dropped
    assert r["levels"] == 2                  # level 2 has no earlier model to compare with; after it nothing moved: stop
    assert (r["level_of"] > 0).sum() == 5


def test_interpolation_at_every_sampled_frequency():
    s, orc, H, plist, B, C = _setup(o=4, v=6, Q=5, seed=12)
    eta = 0.025
    r = workflow.run(H, B, C, -1.4, -0.4, 0.02, eta, spec_tol=1e-4)
    k = np.nonzero(r["level_of"])[0]
    Gd = orc.G_dense(plist, r["w"][k], eta, H)
    assert np.abs(r["G"][k] - Gd).max() < 1e-9 * np.abs(Gd).max()


def test_full_refinement_reproduces_the_dense_spectral_function():
    s, orc, H, plist, B, C = _setup(o=3, v=3, Q=4, seed=9)
    eta = 0.05
    wmin, wmax, dw = -1.6, -0.96, 0.01                  # 65 grid points: 2^6 intervals
    r = workflow.run(H, B, C, wmin, wmax, dw, eta, spec_tol=0.0)
    n = H.shape[0]
    Gd = orc.G_dense(plist, r["w"], eta, H)
    Ad = np.einsum("wpp->w", Gd.imag) / np.pi
    # the subspace saturates (m = n) long before the grid is exhausted: the model IS the full system
    assert r["m"] == n
    assert np.abs(r["A"] - Ad).max() < 1e-9 * np.abs(Ad).max()
