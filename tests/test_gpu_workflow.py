"""GPU parity of the level loop (gfcc_spectral_adaptive) against oracle/workflow.py through the C ABI (-m gpu).

What is unique is compared: the set of sampled grid points per level and the number of levels (integer decisions: both sides
take them from spectral functions that agree to ~1e-9, and the test cases keep the decisive differences far from spec_tol),
the subspace dimension m, and A(omega), G^(omega) on the whole fine grid at north_star's G tolerance (1e-8 relative).
"""
import numpy as np
import pytest
import torch

import oracle
from oracle import workflow
from gfcc_testutil import random_system

pytestmark = pytest.mark.gpu
TOL_G = 1e-8


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def _pair(o, v, Q, seed, t_scale=0.03, l_scale=0.1):
    import paper_2010_04768_b200 as g
    s = random_system(o, v, Q, seed=seed, t_scale=t_scale, l_scale=l_scale)
    orc = oracle.Oracle(o, v, Q, s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"], oracle.MODE_DEF)
    h = g.gfcc_create(o, v, Q, *[dev(s[k]) for k in ("fock", "T1", "T2p", "L1", "L2p", "Lchol")])
    return g, s, orc, h


@pytest.mark.parametrize("o,v,Q,seed,engine", [(4, 5, 6, 31, 0), (6, 10, 8, 11, 0), (5, 8, 7, 3, 1)])
def test_level_loop_matches_oracle(o, v, Q, seed, engine):
    g, s, orc, h = _pair(o, v, Q, seed)
    H = orc.dense_hbar()
    plist = [o - 1, o - 2, o + 1]
    B = np.stack([orc.pack(*orc.rhs(p)).real for p in plist], axis=1)
    C = np.stack([orc.pack(*orc.bra(q)) for q in plist], axis=1)
    wmin, wmax, dw, eta, spec_tol = -1.3, -0.3, 0.02, 0.04, 3e-3
    ref = workflow.run(H, B, C, wmin, wmax, dw, eta, spec_tol=spec_tol)
    g.gfcc_set_option(h, "gmres_m", 400)
    if engine:
        g.gfcc_set_option(h, "engine", 1)
    out = g.gfcc_spectral_adaptive(h, plist, wmin, wmax, dw, eta, 1e-12, spec_tol=spec_tol)
    assert out["levels"] == ref["levels"] and out["m"] == ref["m"]
    assert np.array_equal(out["level_of"], ref["level_of"])
    assert np.abs(out["w"] - ref["w"]).max() < 1e-14
    assert np.abs(out["A"] - ref["A"]).max() < TOL_G * np.abs(ref["A"]).max()
    assert np.abs(out["G"] - ref["G"]).max() < TOL_G * np.abs(ref["G"]).max()
    # Eq. 12 counts on the GPU side too
    lo = out["level_of"]
    assert (lo == 1).sum() == 3
    for L in range(2, out["levels"] + 1):
        assert 1 <= (lo == L).sum() <= 2 ** (L - 1)
    # interpolation: the final model reproduces the unreduced dense G at every sampled frequency
    k = np.nonzero(lo)[0]
    Gd = orc.G_dense(plist, out["w"][k], eta, H)
    assert np.abs(out["G"][k] - Gd).max() < TOL_G * np.abs(Gd).max()
    g.gfcc_destroy(h)


def test_level_loop_caps_and_errors():
    g, s, orc, h = _pair(4, 5, 6, 31)
    plist = [3, 2]
    g.gfcc_set_option(h, "gmres_m", 300)
    out = g.gfcc_spectral_adaptive(h, plist, -0.8, -0.4, 0.01, 0.03, 1e-11, spec_tol=0.0, max_levels=2)
    assert out["levels"] == 2 and (out["level_of"] > 0).sum() == 5 and len(out["w"]) == 41       # Eq. 12: 3 + 2
    out = g.gfcc_spectral_adaptive(h, plist, -0.8, -0.4, 0.01, 0.03, 1e-11, spec_tol=0.0)
    assert out["levels"] <= 5                                                                    # Eq. 13, the paper's own example
    with pytest.raises(g.GfccError):
        g.gfcc_spectral_adaptive(h, plist, -0.4, -0.8, 0.01, 0.03, 1e-11)                         # empty window
    with pytest.raises(g.GfccError):
        g.gfcc_spectral_adaptive(h, [99], -0.8, -0.4, 0.01, 0.03, 1e-11)                          # orbital out of range
    g.gfcc_destroy(h)
