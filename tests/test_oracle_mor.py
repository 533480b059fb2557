"""Pins of the MOR oracle (oracle/mor.py) against things that are NOT the oracle (run with -m "not gpu").

Eq. 10 / Alg. 1 lines 18-21.  What the mathematics fixes:
  (g) S^T S = 1, span(S) contains Re and Im of every sampled X;
  (h) INTERPOLATION: a Galerkin projection onto a space that contains X_p(omega_k) reproduces G(omega_k) exactly;
  (i) FULL SPACE: with m = n the reduced model is the original one at EVERY omega;
  (j) the reduced solve through an eigen-decomposition of H^ (numpy.linalg.eig, a different library route);
  (k) basis invariance: G^ depends on span(S) only (a rotated basis gives the same G^);
  (l) Eq. 9 on the closed form T = Lambda = L = 0: A(omega) = (1/pi) sum_p eta / ((omega - eps_p)^2 + eta^2) >= 0
      (a sum of unit-weight Lorentzians; this fixes the sign reading of Eq. 9 against Eq. 5's -i eta).
"""
import numpy as np

import oracle
from oracle import mor
from gfcc_testutil import random_system


def make_oracle(s):
    return oracle.Oracle(s["o"], s["v"], s["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"], oracle.MODE_DEF)


def _setup(o=4, v=5, Q=6, seed=31):
    s = random_system(o, v, Q, seed=seed, t_scale=0.05, l_scale=0.15)
    orc = make_oracle(s)
    H = orc.dense_hbar()
    plist = [o - 1, o - 2, o + 1]
    B = np.stack([orc.pack(*orc.rhs(p)).real for p in plist], axis=1)
    C = np.stack([orc.pack(*orc.bra(q)) for q in plist], axis=1)
    return s, orc, H, plist, B, C


def _exact_X(H, B, omegas, eta):
    n = H.shape[0]
    return np.concatenate([np.linalg.solve(H + (w - 1j * eta) * np.eye(n), B.astype(np.complex128)).T for w in omegas], axis=0)


def test_mor_orthonormal_and_span():
    s, orc, H, plist, B, C = _setup()
    X = _exact_X(H, B, [-0.9, -0.5, -0.2], 0.02)
    S = mor.mor_extend(None, X, 1e-10)
    assert S.shape[1] == 2 * X.shape[0]                      # generic vectors: nothing dropped
    assert np.abs(S.T @ S - np.eye(S.shape[1])).max() < 1e-13
    for x in X:                                              # Re and Im of every sampled X lie in span(S)
        for part in (x.real, x.imag):
            assert np.linalg.norm(part - S @ (S.T @ part)) < 1e-11 * np.linalg.norm(part)
    # a duplicate is dropped, an extension keeps the old columns
    S2 = mor.mor_extend(S, X[:2], 1e-8)
    assert S2.shape == S.shape and np.array_equal(S2, S)
    S3 = mor.mor_extend(S, _exact_X(H, B, [-0.7], 0.02), 1e-10)
    assert np.array_equal(S3[:, :S.shape[1]], S) and np.abs(S3.T @ S3 - np.eye(S3.shape[1])).max() < 1e-13


def test_mor_interpolates_sampled_frequencies():
    s, orc, H, plist, B, C = _setup()
    eta, ws = 0.02, [-0.9, -0.5, -0.2]
    S = mor.mor_extend(None, _exact_X(H, B, ws, eta), 1e-10)
    Hh, bh, ch = mor.mor_project(H, S, B, C)
    G, A = mor.mor_green(Hh, bh, ch, ws, eta)
    Gref = orc.G_dense(plist, ws, eta, H)
    assert np.abs(G - Gref).max() < 1e-10 * np.abs(Gref).max()
    assert np.abs(A - np.einsum("wpp->w", Gref.imag) / np.pi).max() < 1e-10
    # ... and is only an approximation in between (so the test above is not vacuous)
    S1 = mor.mor_extend(None, _exact_X(H, B, ws[:1], eta), 1e-10)
    G1, _ = mor.mor_green(*mor.mor_project(H, S1, B, C), ws, eta)
    assert np.abs(G1[0] - Gref[0]).max() < 1e-10 * np.abs(Gref).max()       # exact at the one sampled point
    assert np.abs(G1[2] - Gref[2]).max() > 1e-6                              # not elsewhere


def test_mor_full_space_is_exact():
    s, orc, H, plist, B, C = _setup(o=3, v=2, Q=4, seed=5)
    n = H.shape[0]
    rng = np.random.default_rng(3)
    X = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    S = mor.mor_extend(None, X, 1e-8)
    assert S.shape == (n, n)                                 # Im parts are dropped once the space is full
    Hh, bh, ch = mor.mor_project(H, S, B, C)
    ws = np.linspace(-1.1, 0.3, 7)
    G, _ = mor.mor_green(Hh, bh, ch, ws, 0.03)
    Gref = orc.G_dense(plist, ws, 0.03, H)
    assert np.abs(G - Gref).max() < 1e-11 * np.abs(Gref).max()


def test_mor_green_eig_route_and_basis_invariance():
    s, orc, H, plist, B, C = _setup()
    eta = 0.02
    S = mor.mor_extend(None, _exact_X(H, B, [-0.8, -0.3], eta), 1e-10)
    Hh, bh, ch = mor.mor_project(H, S, B, C)
    ws = np.linspace(-1.0, -0.1, 5)
    G, _ = mor.mor_green(Hh, bh, ch, ws, eta)
    lam, V = np.linalg.eig(Hh)
    Vib = np.linalg.solve(V, bh.astype(np.complex128))
    for iw, w in enumerate(ws):
        Gw = ((ch.T @ V) @ (Vib / (w - 1j * eta + lam)[:, None])).T
        assert np.abs(G[iw] - Gw).max() < 1e-10 * np.abs(Gw).max()
    Qrot, _ = np.linalg.qr(np.random.default_rng(1).normal(size=(S.shape[1], S.shape[1])))
    G2, _ = mor.mor_green(*mor.mor_project(H, S @ Qrot, B, C), ws, eta)
    assert np.abs(G2 - G).max() < 1e-10 * np.abs(G).max()


def test_mor_spectral_function_closed_form():
    o, v, Q = 3, 3, 2
    s = random_system(o, v, Q, seed=9, diag_f=True)
    z = lambda a: np.zeros_like(a)
    orc = oracle.Oracle(o, v, Q, s["fock"], z(s["T1"]), z(s["T2p"]), z(s["L1"]), z(s["L2p"]), z(s["Lchol"]), oracle.MODE_DEF)
    H = orc.dense_hbar()
    plist = list(range(o))
    B = np.stack([orc.pack(*orc.rhs(p)).real for p in plist], axis=1)
    C = np.stack([orc.pack(*orc.bra(q)) for q in plist], axis=1)
    eta = 0.05
    S = mor.mor_extend(None, _exact_X(H, B, [-1.3], eta), 1e-10)    # X_p = e_p / (w - eps_p - i eta): m = o after the drops
    assert S.shape[1] == o
    ws = np.linspace(-2.5, -0.5, 9)
    _, A = mor.mor_green(*mor.mor_project(H, S, B, C), ws, eta)
    eps = np.diag(s["fock"])[:o]
    Aref = np.array([np.sum(eta / ((w - eps) ** 2 + eta ** 2)) / np.pi for w in ws])
    assert np.abs(A - Aref).max() < 1e-12 * Aref.max()
