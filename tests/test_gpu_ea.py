"""GPU parity of the EA / advanced part (Eq. 6, second terms of Eq. 7-8) against the CPU
oracle's definition form (oracle.MODE_EA, pinned by the Fock-space brute force in tests/test_oracle_ea.py), through the
C ABI: sigma_EA at 1e-10, G^A at 1e-8 (the tolerances BASELINE.json north_star states for the IP part).  -m gpu."""
import os

import numpy as np
import pytest
import torch

import oracle
from gfcc_testutil import random_system, relmax, to_numpy_system

pytestmark = pytest.mark.gpu

TOL_SIGMA = 1e-10
TOL_G = 1e-8
GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def make_pair(s):
    import paper_2010_04768_b200 as g
    orc = oracle.Oracle(s["o"], s["v"], s["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"],
                        oracle.MODE_DEF | oracle.MODE_EA)
    keep = [dev(s[k]) for k in ("fock", "T1", "T2p", "L1", "L2p", "Lchol")]
    h = g.gfcc_create(s["o"], s["v"], s["Q"], *keep)
    return g, orc, h


def random_y(o, v, nrhs, seed):
    rng = np.random.default_rng(seed)
    y1 = rng.normal(size=(nrhs, v)) + 1j * rng.normal(size=(nrhs, v))
    y2 = rng.normal(size=(nrhs, o, v, v)) + 1j * rng.normal(size=(nrhs, o, v, v))
    return y1, y2 - y2.transpose(0, 1, 3, 2)


@pytest.mark.parametrize("o,v,Q,sym,nrhs", [(2, 2, 1, True, 1), (3, 3, 4, True, 3), (4, 6, 5, False, 2), (5, 7, 9, True, 4),
                                            (12, 37, 50, True, 5), (9, 70, 33, False, 7)])
def test_sigma_ea_small(o, v, Q, sym, nrhs):
    s = random_system(o, v, Q, seed=7 + o + v, sym_L=sym, l_scale=0.3 if o < 9 else 0.1)
    g, orc, h = make_pair(s)
    y1, y2 = random_y(o, v, nrhs, seed=5)
    w = 0.3 + 0.1 * np.arange(nrhs)
    S1, S2 = orc.sigma_ea(w, 0.01, y1, y2)
    G1, G2 = g.gfcc_sigma_ea(h, w, 0.01, dev(y1), dev(y2))
    assert relmax(G1.cpu().numpy(), S1) < TOL_SIGMA and relmax(G2.cpu().numpy(), S2) < TOL_SIGMA
    G2n = G2.cpu().numpy()
    assert np.array_equal(G2n, -G2n.transpose(0, 1, 3, 2))                       # antisymmetric, zero diagonal: bit-level
    T1, T2 = g.gfcc_sigma_ea(h, w + 0.25, 0.01, dev(y1), dev(y2))               # exact shift identity on the GPU path too
    assert relmax((T2 - G2).cpu().numpy(), 0.25 * y2) < 1e-12
    # G^A assembly alone
    ps = list(range(o + v))
    Ga = g.gfcc_assemble_g_ea(h, dev(y1), dev(y2), ps)
    ref = np.array([[orc.bra_dot_ea(*orc.bra_ea(p), y1[r], y2[r]) for p in ps] for r in range(nrhs)])
    assert relmax(Ga, ref) < 1e-12
    g.gfcc_destroy(h)


@pytest.mark.parametrize("o,v,Q,sym", [(3, 3, 4, True), (4, 6, 5, False), (6, 9, 12, True)])
def test_solve_ea_small_vs_dense_lu(o, v, Q, sym):
    s = random_system(o, v, Q, seed=17 + o, sym_L=sym, l_scale=0.2)
    g, orc, h = make_pair(s)
    plist = [o, o + v - 1, 0, o - 1]               # virtual and occupied targets
    ws = [0.3, 0.9, -0.4]
    Gd = orc.G_dense_ea(plist, ws, 0.02)
    g.gfcc_set_option(h, "gmres_m", 500)
    G, Y1, Y2 = g.gfcc_solve_ea(h, plist, ws, 0.02, 1e-11, return_y=True)
    assert relmax(G, Gd) < TOL_G
    # solver-independent: the GPU's Y in the ORACLE's sigma_EA has true residual <= tol
    Y1n, Y2n = Y1.cpu().numpy(), Y2.cpu().numpy()
    wr = np.array([ws[iw] for iq in range(len(plist)) for iw in range(len(ws))])
    S1, S2 = orc.sigma_ea(wr, 0.02, Y1n, Y2n)
    for r in range(len(wr)):
        b1, b2 = orc.rhs_ea(plist[r // len(ws)])
        res = orc.pack_ea(b1 - S1[r], b2 - S2[r])
        assert np.linalg.norm(res) / np.linalg.norm(orc.pack_ea(b1, b2)) < 1e-9
    rel, its = g.gfcc_get_residuals(h, len(wr))
    assert (rel <= 1e-11).all() and (its > 0).all()
    # small batches with refill, zero initial guess: same G
    g.gfcc_set_option(h, "x0", 0)
    g.gfcc_set_option(h, "max_batch", 5)
    G2 = g.gfcc_solve_ea(h, plist, ws, 0.02, 1e-11)
    assert relmax(G2, Gd) < TOL_G
    # the IP part on the same handle is untouched: full GFCCSD matrix element = IP term + EA term (Eq. 8)
    Gip = g.gfcc_solve_ip(h, plist, ws, 0.02, 1e-11)
    orc_ip = orc.G_dense(plist, ws, 0.02)
    assert relmax(Gip + G2, orc_ip + Gd) < TOL_G
    g.gfcc_destroy(h)


def test_config0_ea():
    import gfcc_inputs
    s = to_numpy_system(gfcc_inputs.make_config(0, "cpu"))
    g, orc, h = make_pair(s)
    o, v = 8, 24
    y1, y2 = random_y(o, v, 16, seed=9)
    w = np.linspace(0.1, 1.0, 16)
    S1, S2 = orc.sigma_ea(w, s["eta"], y1, y2)
    G1, G2 = g.gfcc_sigma_ea(h, w, s["eta"], dev(y1), dev(y2))
    assert relmax(G1.cpu().numpy(), S1) < TOL_SIGMA and relmax(G2.cpu().numpy(), S2) < TOL_SIGMA
    plist = [o, o + 1, o - 1]
    ws = [0.1, 0.4]
    Gd = orc.G_dense_ea(plist, ws, s["eta"])
    g.gfcc_set_option(h, "gmres_m", 600)
    g.gfcc_set_option(h, "gmres_maxit", 3000)
    G = g.gfcc_solve_ea(h, plist, ws, s["eta"], 1e-11)
    for iw in range(len(ws)):
        assert np.abs(G[iw] - Gd[iw]).max() <= TOL_G * np.abs(Gd[iw]).max()
    g.gfcc_destroy(h)


def test_config1_ea_vs_definition_form_oracle():
    """config 1 (o=40, v=160, Q=600) at full size against values STORED by tests/golden/make_config1_ea.py (which calls only
    oracle/ and gfcc_inputs/): sigma_EA rows of seeded trial vectors, G^A assembly, and for q = o at omega = -0.4 the GMRES
    residual history, the unique k-step iterate and G^A from it."""
    import gfcc_inputs as gi
    import paper_2010_04768_b200 as g
    gold = np.load(os.path.join(GOLD, "config1_ea.npz"))
    c = gi.CONFIGS[1]
    o, v = c["o"], c["v"]
    s = gi.make_config(1, "cpu")                  # the golden file was written from CPU-drawn inputs: same bits
    h = g.gfcc_create(o, v, c["Q"], *[s[k].cuda() for k in ("fock", "T1", "T2p", "L1", "L2p", "Lchol")])
    nsel = int(gold["nsel"])
    Y1, Y2 = gi.trial_vectors_ea(o, v, nsel, gi.seed_of(1), "cpu")
    Y1, Y2 = Y1.cuda(), Y2.cuda()
    S1, S2 = g.gfcc_sigma_ea(h, gold["omega"], float(gold["eta"]), Y1, Y2)
    S1h, S2h = S1.cpu().numpy(), S2.cpu().numpy()
    e1 = np.abs(S1h[:, gold["s1rows"]].T - gold["S1s"]).max() / float(gold["scale1"])
    e2 = np.abs(np.stack([S2h[:, j, a, b] for (j, a, b) in gold["rows"]]) - gold["S2s"]).max() / float(gold["scale2"])
    assert e1 < TOL_SIGMA and e2 < TOL_SIGMA, (e1, e2)
    Ga = g.gfcc_assemble_g_ea(h, Y1, Y2, gold["plist"])
    assert np.abs(Ga - gold["GA"]).max() <= TOL_G * np.abs(gold["GA"]).max()
    k = int(gold["kfix"])
    g.gfcc_set_option(h, "gmres_fixed", k)
    G, X1, X2 = g.gfcc_solve_ea(h, gold["plist"], [float(gold["om"])], float(gold["eta"]), 1e-30, return_y=True)
    g.gfcc_set_option(h, "gmres_fixed", 0)
    iq = list(gold["plist"]).index(int(gold["q"]))
    hist = g.gfcc_get_residual_history(h, iq)
    assert len(hist) == k + 1 and np.abs(hist / gold["hist"] - 1).max() < 1e-6
    X1h, X2h = X1[iq].cpu().numpy(), X2[iq].cpu().numpy()
    sc = max(np.abs(X1h).max(), np.abs(X2h).max())
    assert np.abs(X1h - gold["Y1k"]).max() <= 1e-8 * sc
    assert np.abs(np.array([X2h[j, a, b] for (j, a, b) in gold["rows"]]) - gold["Y2k"]).max() <= 1e-8 * sc
    assert np.abs(G[0, :, iq] - gold["Gk"]).max() <= TOL_G * np.abs(gold["Gk"]).max()
    g.gfcc_destroy(h)
