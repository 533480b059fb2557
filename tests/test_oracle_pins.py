"""Pins of the CPU oracle against things that are NOT the oracle (run with -m "not gpu").

(e) Fock-space brute force (tests/gfcc_fockspace.py): every block of Hbar_IP, b_p, c_q, G_pq.
(a) closed form at T = Lambda = L = 0:  G_ii(w) = 1/(w - eps_i - i eta), 2h1p diagonal.
(b) linearity, exact shift identity, antisymmetry, Re/Im decoupling, symmetry at T=0, f_ov=0.
(c) sigma from an explicit 4-index <pq||rs> numpy tensor (einsum restatement of SURVEY.md 8c).
(d) GMRES vs dense LU at config 0.
(f) row-sampled factorised sigma == definition-form sigma.
"""
import numpy as np
import pytest

import oracle
import gfcc_fockspace as fockspace
from gfcc_testutil import random_system, random_x, relmax, to_numpy_system


def make_oracle(s, mode=oracle.MODE_DEF):
    return oracle.Oracle(s["o"], s["v"], s["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"], mode)


# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("o,v,Q,sym", [(3, 3, 4, True), (4, 3, 3, False), (3, 4, 5, True), (2, 5, 3, False)])
def test_fockspace_pin(o, v, Q, sym):
    s = random_system(o, v, Q, seed=100 + 7 * o + v, sym_L=sym)
    HIP, bs, cs = fockspace.brute_force(o, v, s["fock"], s["Lchol"], s["T1"], s["t2"], s["L1"], s["l2"])
    orc = make_oracle(s)
    H = orc.dense_hbar()
    assert np.abs(H - HIP).max() < 5e-14
    for p in range(o + v):
        assert np.abs(orc.pack(*orc.rhs(p)).real - bs[p]).max() < 1e-14
        assert np.abs(orc.pack(*orc.bra(p)) - cs[p]).max() < 1e-14
    # G_pq from the literal definition vs oracle's dense route
    w, eta = -0.37, 0.02
    n = H.shape[0]
    X = np.linalg.solve(HIP + (w - 1j * eta) * np.eye(n), bs.T)
    Gref = (cs @ X).T
    G = orc.G_dense(list(range(o + v)), [w], eta)[0]
    assert np.abs(G - Gref).max() < 1e-12


def test_closed_form_zero_coupling():
    # (a) T = Lambda = 0, L = 0, diagonal f
    o, v, Q = 4, 5, 3
    rng = np.random.default_rng(3)
    eps = np.concatenate([-1.5 + rng.random(o), 0.2 + rng.random(v)])
    z = lambda *sh: np.zeros(sh)
    orc = oracle.Oracle(o, v, Q, np.diag(eps), z(o, v), z(o * (o - 1) // 2, v, v), z(o, v),
                        z(o * (o - 1) // 2, v * (v - 1) // 2), z(Q, o + v, o + v))
    eta = 0.013
    ws = [-0.9, -0.31]
    G = orc.G_dense(list(range(o)), ws, eta)
    for iw, w in enumerate(ws):
        expect = np.diag(1.0 / (w - eps[:o] - 1j * eta))
        assert np.abs(G[iw] - expect).max() < 1e-13
    H = orc.dense_hbar()
    d = np.diag(H)
    assert np.abs(H - np.diag(d)).max() == 0.0
    k = o
    for i in range(o):
        assert abs(d[i] + eps[i]) < 1e-15
    for i in range(o):
        for j in range(i + 1, o):
            for a in range(v):
                assert abs(d[k] - (eps[o + a] - eps[i] - eps[j])) < 1e-14
                k += 1
    # GMRES reproduces the closed form too
    x1, x2, nit, rr = orc.gmres(1, ws[0], eta, 1e-12, m=10, x0kind=0)
    assert abs(x1[1] - 1.0 / (ws[0] - eps[1] - 1j * eta)) < 1e-12


def test_sigma_identities():
    # (b)
    o, v, Q = 4, 6, 5
    s = random_system(o, v, Q, seed=11)
    orc = make_oracle(s)
    x1, x2 = random_x(o, v, 3, seed=5)
    eta = 0.01
    w = np.array([-0.5, -0.7, -0.2])
    S1, S2 = orc.sigma(w, eta, x1, x2)
    # antisymmetry of sigma2
    assert np.abs(S2 + S2.transpose(0, 2, 1, 3)).max() < 1e-13
    # shift identity sigma(w) - sigma(w') = (w - w') X, exactly linear in w
    w2 = w + np.array([0.3, -0.1, 1.0])
    T1, T2 = orc.sigma(w2, eta, x1, x2)
    assert np.abs((S1 - T1) - (w - w2)[:, None] * x1).max() < 1e-13
    assert np.abs((S2 - T2) - (w - w2)[:, None, None, None] * x2).max() < 1e-13
    # linearity
    y1, y2 = random_x(o, v, 3, seed=6)
    al = 0.3 - 1.1j
    U1, U2 = orc.sigma(w, eta, y1, y2)
    V1, V2 = orc.sigma(w, eta, x1 + al * y1, x2 + al * y2)
    assert np.abs(V1 - (S1 + al * U1)).max() < 1e-12
    assert np.abs(V2 - (S2 + al * U2)).max() < 1e-12
    # Re/Im decoupling: Hbar X real for real X (omega = eta = 0)
    R1, R2 = orc.sigma(0.0, 0.0, x1.real, x2.real)
    assert np.abs(R1.imag).max() == 0.0 and np.abs(R2.imag).max() == 0.0
    I1, I2 = orc.sigma(0.0, 0.0, 1j * x1.real, 1j * x2.real)
    assert np.abs(I1 - 1j * R1).max() < 1e-14 and np.abs(I2 - 1j * R2).max() < 1e-14


def test_symmetric_at_T0():
    # T = 0 and f_ov = 0  =>  Hbar_IP is the (Hermitian) CI-like matrix: real symmetric
    o, v, Q = 3, 4, 4
    s = random_system(o, v, Q, seed=21)
    f = s["fock"].copy()
    f[:o, o:] = 0.0
    f[o:, :o] = 0.0
    z = np.zeros_like
    orc = oracle.Oracle(o, v, Q, f, z(s["T1"]), z(s["T2p"]), s["L1"], s["L2p"], s["Lchol"])
    H = orc.dense_hbar()
    assert np.abs(H - H.T).max() < 1e-13


# ---------------------------------------------------------------------------------------------
def einsum_hbar_sigma(s, w, eta, x1, x2):
    """(c) independent numpy restatement from an explicit 4-index tensor."""
    o, v = s["o"], s["v"]
    W = fockspace.antisym_integrals(s["Lchol"])
    f, t1, t2 = s["fock"], s["T1"], s["t2"]
    O, V = slice(0, o), slice(o, o + v)
    tau = t2 + np.einsum("ia,jb->ijab", t1, t1) - np.einsum("ib,ja->ijab", t1, t1)
    Fme = f[O, V] + np.einsum("nf,mnef->me", t1, W[O, O, V, V])
    Fmi = f[O, O] + np.einsum("me,ie->mi", f[O, V], t1) + np.einsum("ne,mnie->mi", t1, W[O, O, O, V]) \
        + 0.5 * np.einsum("mnef,inef->mi", W[O, O, V, V], tau)
    Fae = f[V, V] - np.einsum("me,ma->ae", f[O, V], t1) + np.einsum("mf,amef->ae", t1, W[V, O, V, V]) \
        - 0.5 * np.einsum("mnaf,mnef->ae", tau, W[O, O, V, V])
    Wmnij = W[O, O, O, O] + np.einsum("je,mnie->mnij", t1, W[O, O, O, V]) - np.einsum("ie,mnje->mnij", t1, W[O, O, O, V]) \
        + 0.5 * np.einsum("ijef,mnef->mnij", tau, W[O, O, V, V])
    Wmnie = W[O, O, O, V] + np.einsum("if,mnfe->mnie", t1, W[O, O, V, V])
    Wmbej = W[O, V, V, O] + np.einsum("jf,mbef->mbej", t1, W[O, V, V, V]) - np.einsum("nb,mnej->mbej", t1, W[O, O, V, O]) \
        - np.einsum("jnfb,mnef->mbej", t2, W[O, O, V, V]) - np.einsum("jf,nb,mnef->mbej", t1, t1, W[O, O, V, V])
    par = W[O, V, V, O] - np.einsum("njbf,mnef->mbej", t2, W[O, O, V, V])
    Wmbij = W[O, V, O, O] - np.einsum("me,ijbe->mbij", Fme, t2) - np.einsum("nb,mnij->mbij", t1, Wmnij) \
        + 0.5 * np.einsum("mbef,ijef->mbij", W[O, V, V, V], tau)
    A = np.einsum("mnie,jnbe->mbij", W[O, O, O, V], t2)
    B = np.einsum("ie,mbej->mbij", t1, par)
    Wmbij = Wmbij + A - A.transpose(0, 1, 3, 2) + B - B.transpose(0, 1, 3, 2)
    sh = w - 1j * eta
    s1 = sh * x1 - np.einsum("mi,m->i", Fmi, x1) - np.einsum("me,mie->i", Fme, x2) + 0.5 * np.einsum("nmie,mne->i", Wmnie, x2)
    s2 = sh * x2 + np.einsum("ae,ije->ija", Fae, x2)
    Bt = np.einsum("mi,mja->ija", Fmi, x2)
    s2 = s2 - (Bt - Bt.transpose(1, 0, 2)) + np.einsum("maji,m->ija", Wmbij, x1) + 0.5 * np.einsum("mnij,mna->ija", Wmnij, x2)
    R = np.einsum("maei,mje->ija", Wmbej, x2)
    s2 = s2 + R - R.transpose(1, 0, 2) + 0.5 * np.einsum("mnef,mnf,ijae->ija", W[O, O, V, V], x2, t2)
    inter = dict(Fme=Fme, Fmi=Fmi, Fae=Fae, Wmnij=Wmnij, Wmnie=Wmnie, Wmbej=Wmbej, Wmbij=Wmbij)
    return inter, s1, s2


@pytest.mark.parametrize("o,v,Q,sym", [(4, 6, 5, True), (5, 7, 9, False)])
def test_four_index_route(o, v, Q, sym):
    s = random_system(o, v, Q, seed=31 + o, sym_L=sym)
    orc = make_oracle(s)
    x1, x2 = random_x(o, v, 2, seed=8)
    w, eta = np.array([-0.45, -0.8]), 0.01
    S1, S2 = orc.sigma(w, eta, x1, x2)
    for r in range(2):
        inter, e1, e2 = einsum_hbar_sigma(s, w[r], eta, x1[r], x2[r])
        assert relmax(S1[r], e1) < 1e-13
        assert relmax(S2[r], e2) < 1e-13
    for k, val in inter.items():
        assert relmax(orc.get(k), val) < 1e-13, k


# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("o,v,Q,sym", [(4, 6, 5, True), (6, 9, 11, False)])
def test_sampled_rows_equal_definition(o, v, Q, sym):
    # (f): T1-dressed, L-factorised row-sampled sigma == definition form
    s = random_system(o, v, Q, seed=41 + o, sym_L=sym)
    orc = make_oracle(s, oracle.MODE_DEF | oracle.MODE_ROWS)
    x1, x2 = random_x(o, v, 3, seed=9)
    w, eta = np.array([-0.45, -0.8, -0.3]), 0.02
    S1, S2 = orc.sigma(w, eta, x1, x2)
    rng = np.random.default_rng(2)
    trip = np.stack([rng.integers(0, o, 12), rng.integers(0, o, 12), rng.integers(0, v, 12)], axis=1)
    trip[0] = (1, 1, 2)      # diagonal pair: must give zero
    R1, R2 = orc.sigma_rows(w, eta, x1, x2, np.arange(o), trip)
    assert relmax(R1, S1.T) < 1e-13
    ref = np.stack([S2[:, i, j, a] for (i, j, a) in trip])
    assert np.abs(R2 - ref).max() / np.abs(S2).max() < 1e-13
    assert np.abs(R2[0]).max() < 1e-13


# ---------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def cfg0():
    import gfcc_inputs
    s = to_numpy_system(gfcc_inputs.make_config(0, "cpu"))
    orc = make_oracle(s, oracle.MODE_DEF | oracle.MODE_ROWS)
    return s, orc, orc.dense_hbar()


def test_config0_gmres_vs_dense_lu(cfg0):
    # (d) config 0: 680 x 680 dense LU vs per-RHS GMRES
    s, orc, H = cfg0
    n = H.shape[0]
    assert n == 8 + 28 * 24
    eta = s["eta"]
    tg = s["targets"]
    ws = [float(s["omegas"][0]), float(s["omegas"][5])]
    G = orc.G_dense(tg, ws, eta, H)
    for iw, w in enumerate(ws):
        for ip, p in enumerate(tg[:2]):
            x1, x2, nit, rr = orc.gmres(p, w, eta, 1e-11, m=300, maxit=2000, x0kind=1)
            assert rr <= 1e-11
            xs = np.linalg.solve(H + (w - 1j * eta) * np.eye(n), orc.pack(*orc.rhs(p)))
            assert relmax(orc.pack(x1, x2), xs) < 1e-8
            for iq, q in enumerate(tg):
                g = orc.bra_dot(*orc.bra(q), x1, x2)
                assert abs(g - G[iw, ip, iq]) <= 1e-8 * np.abs(G[iw]).max()
    # restarted GMRES and x0 = 0 reach the same solution
    x1, x2, nit, rr = orc.gmres(tg[0], ws[1], eta, 1e-10, m=40, maxit=5000, x0kind=0)
    xs = np.linalg.solve(H + (ws[1] - 1j * eta) * np.eye(n), orc.pack(*orc.rhs(tg[0])))
    assert rr <= 1e-10 and relmax(orc.pack(x1, x2), xs) < 1e-7


def test_config0_gmres_residual_history_is_the_krylov_minimum(cfg0):
    """the residual history returned by the oracle GMRES (used to check the GPU solver step by step) against the DEFINITION
    of GMRES: after k steps the residual norm is min over the Krylov space span{r0, A r0, ..} of ||r0 - A z||, here from a
    dense least-squares solve with the assembled 680 x 680 matrix; hist[0] is ||b - A x0|| / ||b||."""
    s, orc, H = cfg0
    n = H.shape[0]
    eta, p, w = s["eta"], s["targets"][1], float(s["omegas"][3])
    A = H + (w - 1j * eta) * np.eye(n)
    b = orc.pack(*orc.rhs(p))
    f = np.diag(np.asarray(s["fock"]))
    o, v = 8, 24
    iu = np.triu_indices(o, 1)
    d = np.concatenate([-f[:o], (f[o:][None, :] - f[iu[0]][:, None] - f[iu[1]][:, None]).reshape(-1)])
    x0 = b / (w - 1j * eta + d)
    r0 = b - A @ x0
    kmax = 12
    x1, x2, nit, rr, hist = orc.gmres(p, w, eta, 1e-30, m=kmax, maxit=kmax + 1, x0kind=1, history=True)
    assert nit == kmax + 1 and len(hist) == kmax + 1
    bn = np.linalg.norm(b)
    assert abs(hist[0] - np.linalg.norm(r0) / bn) < 1e-12 * hist[0]
    K = [r0 / np.linalg.norm(r0)]
    for k in range(1, kmax + 1):
        Kq, _ = np.linalg.qr(np.stack(K, axis=1))
        AK = A @ Kq
        y = np.linalg.lstsq(AK, r0, rcond=None)[0]
        ref = np.linalg.norm(r0 - AK @ y) / bn
        assert abs(hist[k] - ref) < 1e-9 * ref, (k, hist[k], ref)
        nxt = A @ Kq[:, -1]
        K.append(nxt / np.linalg.norm(nxt))
    assert (np.diff(hist) <= 1e-15).all()                      # monotone, PAPER.md:136 ("the residual norm decreases monotonically")
    assert rr == hist[-1]


def test_config0_rows_and_physics(cfg0):
    s, orc, H = cfg0
    import gfcc_inputs
    X1, X2 = gfcc_inputs.trial_vectors(8, 24, 4, gfcc_inputs.seed_of(0))
    X1, X2 = X1.numpy(), X2.numpy()
    w = np.array([-1.0, -0.7, -0.4, -0.2])
    S1, S2 = orc.sigma(w, 0.01, X1, X2)
    trip = np.array([[0, 7, 23], [3, 2, 0], [6, 7, 11], [5, 1, 17]])
    R1, R2 = orc.sigma_rows(w, 0.01, X1, X2, np.arange(8), trip)
    assert relmax(R1, S1.T) < 1e-13
    ref = np.stack([S2[:, i, j, a] for (i, j, a) in trip])
    assert np.abs(R2 - ref).max() / np.abs(S2).max() < 1e-13
    # the synthetic spectrum is what SURVEY.md 8c-13 says: shifted matrices stay regular only through eta
    ev = np.linalg.eigvals(H)
    assert np.isfinite(ev).all() and ev.real.max() < 20.0


def test_sampled_rows_equal_definition_at_config1():
    """the row-sampled (T1-dressed, factorised) oracle -- the only sigma checker at configs 1-4 -- against the DEFINITION form
    at o = 40, v = 160, Q = 600: definition-form values stored by tests/golden/make_config1_def.py (18 minutes of plain loops),
    row-sampled values computed here.  An indexing slip that only shows above the tiny sizes of the other pins fails this one."""
    import os
    import gfcc_inputs as gi
    gold = np.load(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config1_def.npz"))
    c = gi.CONFIGS[1]
    o, v = c["o"], c["v"]
    s = gi.make_config(1, "cpu")
    orc = oracle.Oracle(o, v, c["Q"], *[s[k].numpy() for k in ("fock", "T1", "T2p", "L1", "L2p", "Lchol")], oracle.MODE_ROWS)
    nrhs = int(gold["nrhs"])
    X1, X2 = gi.trial_vectors(o, v, nrhs, gi.seed_of(1), "cpu")
    rsel = [int(r) for r in gold["rsel"]]
    R1, R2 = orc.sigma_rows(gold["omega"][rsel], c["eta"], X1[rsel].numpy(), X2[rsel].numpy(), gold["s1rows"], gold["trip"])
    assert np.abs(R1 - gold["S1def"]).max() < 1e-12 * np.abs(gold["S1def"]).max()
    assert np.abs(R2 - gold["S2def"]).max() < 1e-12 * np.abs(gold["S2def"]).max()
