"""Pins of the oracle's EA / advanced part (Eq. 4, Eq. 6, second terms of
Eq. 7-8) against things that are NOT the oracle (run with -m "not gpu"):
  Fock-space brute force (tests/gfcc_fockspace.py: Jordan-Wigner matrices, Hbar = exp(-T) H_N exp(T), basis tau_a = a+_a,
  tau_jab = a+_a a+_b a_j): every block of Hbar_EA, b_q, c_p, G^A_pq;  closed form 1/(omega - eps_a + i eta);
  exact shift identity, linearity, antisymmetry, Re/Im decoupling; GMRES vs dense LU; symmetry at T = 0, f_ov = 0."""
import numpy as np
import pytest

import oracle
import gfcc_fockspace as fockspace
from gfcc_testutil import random_system, relmax


def make_oracle(s):
    return oracle.Oracle(s["o"], s["v"], s["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"],
                         oracle.MODE_DEF | oracle.MODE_EA)


def random_y(o, v, nrhs, seed):
    rng = np.random.default_rng(seed)
    y1 = rng.normal(size=(nrhs, v)) + 1j * rng.normal(size=(nrhs, v))
    y2 = rng.normal(size=(nrhs, o, v, v)) + 1j * rng.normal(size=(nrhs, o, v, v))
    return y1, y2 - y2.transpose(0, 1, 3, 2)


@pytest.mark.parametrize("o,v,Q,sym", [(2, 3, 4, True), (3, 3, 3, False), (2, 4, 5, False), (3, 4, 4, True)])
def test_fockspace_pin_ea(o, v, Q, sym):
    s = random_system(o, v, Q, seed=200 + 7 * o + v, sym_L=sym)
    HEA, bs, cs = fockspace.brute_force_ea(o, v, s["fock"], s["Lchol"], s["T1"], s["t2"], s["L1"], s["l2"])
    orc = make_oracle(s)
    H = orc.dense_hbar_ea()
    assert np.abs(H - HEA).max() < 5e-14
    for p in range(o + v):
        assert np.abs(orc.pack_ea(*orc.rhs_ea(p)).real - bs[p]).max() < 1e-14
        assert np.abs(orc.pack_ea(*orc.bra_ea(p)) - cs[p]).max() < 1e-14
    # G^A_pq from the literal definition (second term of Eq. 2) vs the oracle's dense route
    w, eta = 0.41, 0.02
    n = H.shape[0]
    Y = np.linalg.solve((w + 1j * eta) * np.eye(n) - HEA, bs.T)
    Gref = cs @ Y                                    # [p, q]
    G = orc.G_dense_ea(list(range(o + v)), [w], eta)[0]
    assert np.abs(G - Gref).max() < 1e-12 * max(1.0, np.abs(Gref).max())      # omega may sit next to a pole of the random system
    # bra_dot_ea is the packed (a<b) dot product
    y1, y2 = random_y(o, v, 1, 3)
    c1, c2 = orc.bra_ea(o)
    assert abs(orc.bra_dot_ea(c1, c2, y1[0], y2[0]) - orc.pack_ea(c1, c2) @ orc.pack_ea(y1[0], y2[0])) < 1e-13


def test_closed_form_zero_coupling_ea():
    o, v, Q = 3, 4, 2
    rng = np.random.default_rng(5)
    eps = np.concatenate([-1.5 + rng.random(o), 0.2 + rng.random(v)])
    z = lambda *sh: np.zeros(sh)
    orc = oracle.Oracle(o, v, Q, np.diag(eps), z(o, v), z(o * (o - 1) // 2, v, v), z(o, v),
                        z(o * (o - 1) // 2, v * (v - 1) // 2), z(Q, o + v, o + v), oracle.MODE_DEF | oracle.MODE_EA)
    eta = 0.017
    ws = [0.3, 1.1]
    virt = list(range(o, o + v))
    G = orc.G_dense_ea(virt, ws, eta)
    for iw, w in enumerate(ws):
        assert np.abs(G[iw] - np.diag(1.0 / (w - eps[o:] + 1j * eta))).max() < 1e-13       # G^A_aa = 1/(omega - eps_a + i eta)
    H = orc.dense_hbar_ea()
    d = np.diag(H)
    assert np.abs(H - np.diag(d)).max() == 0.0
    k = v
    for a in range(v):
        assert abs(d[a] - eps[o + a]) < 1e-15
    for j in range(o):
        for a in range(v):
            for b in range(a + 1, v):
                assert abs(d[k] - (eps[o + a] + eps[o + b] - eps[j])) < 1e-14
                k += 1
    y1, y2, nit, rr = orc.gmres_ea(o + 1, ws[0], eta, 1e-12, m=10, x0kind=0)
    assert abs(y1[1] - 1.0 / (ws[0] - eps[o + 1] + 1j * eta)) < 1e-12
    # occupied targets have no 1p / 2p1h component at T = 0
    assert np.abs(orc.G_dense_ea([0, 1], ws, eta)).max() == 0.0


def test_sigma_ea_identities():
    o, v, Q = 3, 5, 4
    s = random_system(o, v, Q, seed=31, sym_L=False)
    orc = make_oracle(s)
    y1, y2 = random_y(o, v, 3, 1)
    w = np.array([0.2, 0.5, -0.1])
    S1, S2 = orc.sigma_ea(w, 0.03, y1, y2)
    assert np.abs(S2 + S2.transpose(0, 1, 3, 2)).max() == 0.0 or np.abs(S2 + S2.transpose(0, 1, 3, 2)).max() < 1e-14
    T1, T2 = orc.sigma_ea(w + 0.37, 0.03, y1, y2)
    assert relmax(T1 - S1, 0.37 * y1) < 1e-13 and relmax(T2 - S2, 0.37 * y2) < 1e-13            # exact shift identity
    E1, E2 = orc.sigma_ea(w, 0.0, y1, y2)
    assert relmax(S1 - E1, 0.03j * y1) < 1e-13 and relmax(S2 - E2, 0.03j * y2) < 1e-13          # + i eta (Eq. 6), not - i eta
    a, b = 0.7 - 0.2j, -1.3 + 0.4j
    L1, L2 = orc.sigma_ea(w[:1], 0.03, a * y1[:1] + b * y1[1:2], a * y2[:1] + b * y2[1:2])
    A1, A2 = orc.sigma_ea(np.repeat(w[:1], 2), 0.03, y1[:2], y2[:2])
    assert relmax(L1[0], a * A1[0] + b * A1[1]) < 1e-13 and relmax(L2[0], a * A2[0] + b * A2[1]) < 1e-13
    R1, R2 = orc.sigma_ea(0.0, 0.0, y1.real, y2.real)
    assert np.abs(R1.imag).max() == 0.0 and np.abs(R2.imag).max() == 0.0                        # Hbar real


def test_symmetric_at_T0_ea():
    o, v, Q = 3, 4, 5
    s = random_system(o, v, Q, seed=41, sym_L=True)
    f = s["fock"].copy()
    f[:o, o:] = 0.0
    f[o:, :o] = 0.0
    z = lambda *sh: np.zeros(sh)
    orc = oracle.Oracle(o, v, Q, f, z(o, v), z(o * (o - 1) // 2, v, v), s["L1"], s["L2p"], s["Lchol"],
                        oracle.MODE_DEF | oracle.MODE_EA)
    H = orc.dense_hbar_ea()
    assert np.abs(H - H.T).max() < 1e-13


def test_gmres_ea_vs_dense_lu():
    o, v, Q = 4, 7, 6
    s = random_system(o, v, Q, seed=51, sym_L=True, l_scale=0.2)
    orc = make_oracle(s)
    H = orc.dense_hbar_ea()
    n = H.shape[0]
    eta = 0.02
    plist = [o, o + 3, 1]
    ws = [0.2, -0.6]
    G = orc.G_dense_ea(plist, ws, eta, H)
    for iw, w in enumerate(ws):
        for iq, q in enumerate(plist):
            y1, y2, nit, rr, hist = orc.gmres_ea(q, w, eta, 1e-11, m=400, maxit=2000, x0kind=1, history=True)
            assert rr <= 1e-11 and (np.diff(hist) <= 1e-15).all()
            ys = np.linalg.solve((w + 1j * eta) * np.eye(n) - H, orc.pack_ea(*orc.rhs_ea(q)))
            assert relmax(orc.pack_ea(y1, y2), ys) < 1e-8
            for ip, p in enumerate(plist):
                g = orc.bra_dot_ea(*orc.bra_ea(p), y1, y2)
                assert abs(g - G[iw, ip, iq]) <= 1e-8 * np.abs(G[iw]).max()
