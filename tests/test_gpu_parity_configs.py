"""GPU parity at BASELINE.json's full sizes (run with -m gpu on a B200).

The definition-form oracle needs O(o v^3) memory and O(o^3 v^3) work, so from config 1 upwards the CUDA path is compared
with the ROW-SAMPLED oracle (oracle.MODE_ROWS: exact sigma1[i] and sigma2[i,j,a] at chosen rows through L-factorised sums;
its equality with the definition form is pinned in tests/test_oracle_pins.py).  Inputs are materialised once (on the GPU,
seeded) and the same bits are handed to both sides.  Launch configuration = the one bench.py times: the config's RHS batch,
default panel size, handle options untouched.

Configs 3 and 4 need 30 / 100 GB of host memory and minutes of oracle time per row; they run only with GFCC_TEST_LARGE=1
(the outcome of such a run is recorded in profiles/).
"""
import os

import numpy as np
import pytest
import torch

import gfcc_inputs as gi
import oracle
from gfcc_testutil import relmax

pytestmark = pytest.mark.gpu

TOL_SIGMA = 1e-10
TOL_G = 1e-8


def _setup(cfg):
    import paper_2010_04768_b200 as g
    c = gi.CONFIGS[cfg]
    s = gi.make_config(cfg, "cuda")
    host = {k: s[k].cpu().numpy() for k in ("fock", "T1", "T2p", "L1", "L2p", "Lchol")}
    h = g.gfcc_create(c["o"], c["v"], c["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"])
    del s["Lchol"]
    torch.cuda.empty_cache()                     # hand the 14 GB of Lchol (config 4) back to the driver, not to torch's cache
    orc = oracle.Oracle(c["o"], c["v"], c["Q"], host["fock"], host["T1"], host["T2p"], host["L1"], host["L2p"], host["Lchol"],
                        oracle.MODE_ROWS)
    return g, c, s, h, orc


def _triples(o, v, n, seed):
    """(i<j, a) samples: the corners of the index ranges plus random interior rows."""
    fixed = [(0, 1, 0), (0, o - 1, v - 1), (o - 2, o - 1, v // 2), (1, o // 2, 1)]
    rng = np.random.default_rng(seed)
    out = list(fixed)
    while len(out) < n:
        i, j = sorted(rng.choice(o, 2, replace=False))
        out.append((int(i), int(j), int(rng.integers(0, v))))
    return np.array(out[:n], dtype=np.int32)


def _sampled_sigma_check(cfg, nrhs, rsel, ntrip, s1rows, engine=0):
    g, c, s, h, orc = _setup(cfg)
    o, v = c["o"], c["v"]
    if engine:                                   # INT8 tensor-core engine instead of the graded FP64 DMMA engine
        g.gfcc_set_option(h, "engine", 1)
        g.gfcc_set_option(h, "panel_bytes", 4.2e9)
    X1, X2 = gi.trial_vectors(o, v, nrhs, gi.seed_of(cfg), "cuda")
    w = np.resize(np.linspace(c["wlo"], c["whi"], c["nw"]), nrhs)
    S1, S2 = g.gfcc_sigma_ip(h, w, c["eta"], X1, X2)
    torch.cuda.synchronize()
    trip = _triples(o, v, ntrip, 100 + cfg)
    X1h, X2h = X1[rsel].cpu().numpy(), X2[rsel].cpu().numpy()
    R1, R2 = orc.sigma_rows(w[rsel], c["eta"], X1h, X2h, s1rows, trip)        # [rows, len(rsel)]
    S1h = S1[rsel].cpu().numpy()
    S2h = S2[rsel].cpu().numpy()
    scale2 = float(S2.abs().max().item())
    scale1 = float(S1.abs().max().item())
    G1 = S1h[:, s1rows].T
    G2 = np.stack([S2h[:, i, j, a] for (i, j, a) in trip], axis=0)
    e1 = np.abs(G1 - R1).max() / scale1
    e2 = np.abs(G2 - R2).max() / scale2
    # antisymmetric partner and the diagonal, bit-exact
    G2t = np.stack([S2h[:, j, i, a] for (i, j, a) in trip], axis=0)
    assert np.array_equal(G2t, -G2)
    assert float(S2[:, torch.arange(o), torch.arange(o), :].abs().max().item()) == 0.0
    if engine:
        assert g.gfcc_get_stat(h, "oz_gemms") > 0 and g.gfcc_get_stat(h, "oz_fail") == 0
    g.gfcc_destroy(h)
    assert e1 < TOL_SIGMA and e2 < TOL_SIGMA, (e1, e2)
    return e1, e2


def test_config1_sigma_sampled_rows():
    """config 1 (o=40, v=160, Q=600): one 64-RHS batch of the 256, 16 sigma2 rows + 4 sigma1 rows x 3 RHS"""
    _sampled_sigma_check(1, 64, [0, 17, 63], 16, [0, 7, 38, 39])


def test_config2_sigma_sampled_rows():
    """config 2 (o=80, v=320, Q=1200): the 64-RHS batch bench.py --config 2 times, 5 sigma2 rows + 2 sigma1 rows x 2 RHS"""
    _sampled_sigma_check(2, 64, [5, 62], 5, [0, 79])


def test_config1_solve_residual_rows_and_G():
    """config 1 solve: converged batched GMRES; the GPU's X is checked WITHOUT the GPU's own sigma: sampled rows of
    b - sigma_oracle(X) are below tol*||b||, and G equals the oracle's bra vectors dotted with X (G assembly at full size)."""
    g, c, s, h, orc = _setup(1)
    o, v = c["o"], c["v"]
    plist = [o - 1, o - 2, o + 3]                 # two occupied targets and one virtual
    # omega above every pole of the synthetic H-bar: with BASELINE.json's coupling strength (||ring block|| ~ 1 Ha) the
    # shifted operator is indefinite inside the config's own window [-1.2, -0.2] and unpreconditioned GMRES (the
    # paper's solver) stagnates there (measured on B200: relres > 1 after 600 steps for every omega
    # <= 0, 400-440 steps to 1e-9 at omega = +0.3; DESIGN.md section 2 reading 23).  sigma itself is checked inside
    # the window by the tests above; this test checks the SOLVER + G assembly at full config-1 size.
    ws = np.array([0.4, 0.5])
    tol = 1e-9
    g.gfcc_set_option(h, "gmres_m", 700)
    g.gfcc_set_option(h, "gmres_maxit", 700)
    G, X1, X2 = g.gfcc_solve_ip(h, plist, ws, c["eta"], tol, return_x=True)
    nr = len(plist) * len(ws)
    rel, its = g.gfcc_get_residuals(h, nr)
    assert (rel <= tol).all() and (its >= 1).all()
    X1h, X2h = X1.cpu().numpy(), X2.cpu().numpy()
    wr = np.array([ws[iw] for ip in range(len(plist)) for iw in range(len(ws))])
    trip = _triples(o, v, 8, 7)
    s1rows = [0, o - 2, o - 1]
    R1, R2 = orc.sigma_rows(wr, c["eta"], X1h, X2h, s1rows, trip)
    for r in range(nr):
        b1, b2 = orc.rhs(plist[r // len(ws)])
        bn = np.linalg.norm(orc.pack(b1, b2))
        res1 = np.abs(b1[s1rows] - R1[:, r]).max()
        res2 = np.abs(np.array([b2[i, j, a] for (i, j, a) in trip]) - R2[:, r]).max()
        assert res1 <= 10 * tol * bn and res2 <= 10 * tol * bn, (r, res1, res2)
    # G assembly vs the oracle's bra vectors on the same X
    for iq, q in enumerate(plist):
        c1, c2 = orc.bra(q)
        for ip in range(len(plist)):
            for iw in range(len(ws)):
                r = ip * len(ws) + iw
                ref = orc.bra_dot(c1, c2, X1h[r], X2h[r])
                assert abs(G[iw, ip, iq] - ref) <= TOL_G * max(abs(ref), np.abs(G[iw]).max())
    g.gfcc_destroy(h)


@pytest.mark.skipif(os.environ.get("GFCC_TEST_LARGE", "0") != "1", reason="set GFCC_TEST_LARGE=1 (needs >100 GB host memory, ~15 min)")
@pytest.mark.parametrize("cfg,ntrip", [(3, 3), (4, 2)])
def test_large_config_sigma_sampled_rows(cfg, ntrip):
    c = gi.CONFIGS[cfg]
    _sampled_sigma_check(cfg, c["np"] * c["nw"], [c["np"] * c["nw"] - 1], ntrip, [c["o"] - 1])


@pytest.mark.skipif(os.environ.get("GFCC_TEST_LARGE", "0") != "1", reason="set GFCC_TEST_LARGE=1 (needs >100 GB host memory, ~15 min)")
@pytest.mark.parametrize("cfg,nrhs,ntrip", [(3, 32, 3), (4, 8, 2)])
def test_large_config_sigma_sampled_rows_engine_ozaki(cfg, nrhs, ntrip):
    """the INT8 tensor-core engine at full size (config 4 with an 8-RHS batch: its extra 20 GB of digit slices beside the 16-RHS
    batch, the borrowed T2/Lambda2 and this test's own X and sigma copies would not fit 180 GB)"""
    c = gi.CONFIGS[cfg]
    _sampled_sigma_check(cfg, nrhs, [nrhs - 1], ntrip, [c["o"] - 1], engine=1)
