"""GPU parity of the MOR calls (gfcc_mor_reset / _extend / _solve) against oracle/mor.py, through the C ABI (-m gpu).

What is unique is compared element by element: the reduced Green's function G^ and the spectral function A (they depend
on span(S) only), the dimension m, and the projector S S^T; the basis vectors themselves are unique up to rounding-level
drop decisions, so they are checked through orthonormality and span.  Tolerance on G^: 1e-8 relative (north_star's G bar).
"""
import numpy as np
import pytest
import torch

import oracle
from oracle import mor
from gfcc_testutil import random_system, relmax

pytestmark = pytest.mark.gpu
TOL_G = 1e-8


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def _pair(o, v, Q, seed, t_scale=0.05, l_scale=0.15):
    import paper_2010_04768_b200 as g
    s = random_system(o, v, Q, seed=seed, t_scale=t_scale, l_scale=l_scale)
    orc = oracle.Oracle(o, v, Q, s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"], oracle.MODE_DEF)
    keep = [dev(s[k]) for k in ("fock", "T1", "T2p", "L1", "L2p", "Lchol")]
    h = g.gfcc_create(o, v, Q, *keep)
    return g, s, orc, h


def _exact_X(orc, H, plist, omegas, eta):
    """oracle solutions X_p(omega) by dense LU: packed (k, n) and ABI-layout (X1 [k,o], X2 [k,o,o,v]); order w-major."""
    n = H.shape[0]
    B = np.stack([orc.pack(*orc.rhs(p)).real for p in plist], axis=1)
    Xp = np.concatenate([np.linalg.solve(H + (w - 1j * eta) * np.eye(n), B.astype(np.complex128)).T for w in omegas], axis=0)
    X1 = np.stack([orc.unpack(x)[0] for x in Xp])
    X2 = np.stack([orc.unpack(x)[1] for x in Xp])
    return Xp, X1, X2


@pytest.mark.parametrize("o,v,Q,seed", [(4, 5, 6, 31), (6, 9, 10, 7), (5, 16, 12, 3)])
def test_mor_extend_and_solve_match_oracle(o, v, Q, seed):
    g, s, orc, h = _pair(o, v, Q, seed)
    H = orc.dense_hbar()
    n = H.shape[0]
    plist = [o - 1, o - 2, o + 1]
    eta = 0.02
    Bm = np.stack([orc.pack(*orc.rhs(p)).real for p in plist], axis=1)
    Cm = np.stack([orc.pack(*orc.bra(q)) for q in plist], axis=1)
    g.gfcc_mor_reset(h, 64)
    S_o = None
    # two levels (Alg. 1: the subspace grows level by level); the second one repeats a sampled frequency -> drops
    for lvl, ws in enumerate(([-0.9, -0.2], [-0.5, -0.9])):
        Xp, X1, X2 = _exact_X(orc, H, plist, ws, eta)
        S_o = mor.mor_extend(S_o, Xp, 1e-8)
        m = g.gfcc_mor_extend(h, dev(X1), dev(X2), 1e-8)
        assert m == S_o.shape[1] == g.gfcc_mor_get(h, "m")
        S_g = g.gfcc_mor_get(h, "S")
        assert S_g.shape == (n, m)
        assert np.abs(S_g.T @ S_g - np.eye(m)).max() < 1e-13                       # orthonormal
        assert np.abs(S_g @ S_g.T - S_o @ S_o.T).max() < 1e-9                      # same span (projector is unique)
        HS = g.gfcc_mor_get(h, "HS")
        assert relmax(HS, H @ S_g) < 1e-10                                         # projection operand = Hbar S
        Hh = g.gfcc_mor_get(h, "Hhat")
        assert relmax(Hh, S_g.T @ (H @ S_g)) < 1e-10
    assert 12 < g.gfcc_mor_get(h, "m") <= 18                                       # 12 + at most 6: the repeated frequency is dropped
    wf = np.linspace(-1.1, 0.1, 25)
    G_g, A_g = g.gfcc_mor_solve(h, plist, wf, eta)
    G_o, A_o = mor.mor_green(*mor.mor_project(H, S_o, Bm, Cm), wf, eta)
    assert np.abs(G_g - G_o).max() < TOL_G * np.abs(G_o).max()
    assert np.abs(A_g - A_o).max() < TOL_G * np.abs(A_o).max()
    # interpolation at a sampled frequency against the UNREDUCED dense solve (Eq. 10 vs Eq. 5)
    G_s, _ = g.gfcc_mor_solve(h, plist, [-0.5], eta)
    G_d = orc.G_dense(plist, [-0.5], eta, H)
    assert np.abs(G_s - G_d).max() < TOL_G * np.abs(G_d).max()
    g.gfcc_destroy(h)


def test_mor_from_gpu_solutions_full_workflow():
    """Alg. 1 end to end on the device: gfcc_solve_ip_x -> gfcc_mor_extend -> gfcc_mor_solve; the reduced model reproduces
    the directly solved G at the sampled frequencies and the oracle's dense G in between within the model error."""
    o, v, Q = 6, 10, 8
    g, s, orc, h = _pair(o, v, Q, 11, t_scale=0.03, l_scale=0.1)
    H = orc.dense_hbar()
    plist = [o - 1, o - 2]
    eta = 0.03
    ws = np.array([-1.0, -0.6, -0.2])
    g.gfcc_set_option(h, "gmres_m", 400)
    G, X1, X2 = g.gfcc_solve_ip(h, plist, ws, eta, 1e-12, return_x=True)
    g.gfcc_mor_reset(h, 40)
    m = g.gfcc_mor_extend(h, X1, X2, 1e-8)
    assert m == 12
    G_m, A_m = g.gfcc_mor_solve(h, plist, ws, eta)
    assert np.abs(G_m - G).max() < 1e-8 * np.abs(G).max()
    assert np.abs(A_m - np.einsum("wpp->w", G.imag) / np.pi).max() < 1e-8 * np.abs(A_m).max()
    wf = np.linspace(-1.0, -0.2, 9)
    G_f, _ = g.gfcc_mor_solve(h, plist, wf, eta)
    G_d = orc.G_dense(plist, wf, eta, H)
    # reduced model built from the same X (oracle side) has the same in-between values
    Xp = np.stack([orc.pack(X1[r].cpu().numpy(), X2[r].cpu().numpy()) for r in range(X1.shape[0])])
    Bm = np.stack([orc.pack(*orc.rhs(p)).real for p in plist], axis=1)
    Cm = np.stack([orc.pack(*orc.bra(q)) for q in plist], axis=1)
    G_o, _ = mor.mor_green(*mor.mor_project(H, mor.mor_extend(None, Xp, 1e-8), Bm, Cm), wf, eta)
    assert np.abs(G_f - G_o).max() < 1e-8 * np.abs(G_o).max()
    assert np.abs(G_f - G_d).max() < 0.2 * np.abs(G_d).max()      # a 12-dimensional model of a 96-dimensional system
    g.gfcc_destroy(h)


def test_mor_edge_cases():
    import paper_2010_04768_b200 as g
    o, v, Q = 3, 2, 3
    gg, s, orc, h = _pair(o, v, Q, 5)
    n = o + o * (o - 1) // 2 * v
    X1 = torch.zeros((1, o), dtype=torch.complex128, device="cuda")
    X2 = torch.zeros((1, o, o, v), dtype=torch.complex128, device="cuda")
    with pytest.raises(g.GfccError):                  # no subspace yet
        g.gfcc_mor_extend(h, X1, X2)
    with pytest.raises(g.GfccError):
        g.gfcc_mor_solve(h, [0], [-0.5], 0.01)
    g.gfcc_mor_reset(h, 1000)                         # capacity is clipped to the dimension (rounded up to even)
    assert g.gfcc_mor_get(h, "cap") in (n, n + 1)
    assert g.gfcc_mor_extend(h, X1, X2) == 0          # zero vectors are dropped, not divided by zero
    with pytest.raises(g.GfccError):                  # still empty
        g.gfcc_mor_solve(h, [0], [-0.5], 0.01)
    # fill the whole space with random vectors: m = n, later candidates are dropped, reduced model == full model
    rng = np.random.default_rng(2)
    Xp = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    X1 = dev(np.stack([orc.unpack(x)[0] for x in Xp]))
    X2 = dev(np.stack([orc.unpack(x)[1] for x in Xp]))
    assert g.gfcc_mor_extend(h, X1, X2, 1e-8) == n
    plist = [0, o - 1, o]
    wf = np.linspace(-1.5, 0.5, 5)
    G_g, _ = g.gfcc_mor_solve(h, plist, wf, 0.05)
    G_d = orc.G_dense(plist, wf, 0.05)
    assert np.abs(G_g - G_d).max() < 1e-9 * np.abs(G_d).max()
    g.gfcc_mor_reset(h, 0)                            # frees
    assert g.gfcc_mor_get(h, "m") == 0
    g.gfcc_destroy(h)
