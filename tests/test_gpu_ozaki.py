"""GPU parity of the INT8 tensor-core (Ozaki) engine (-m gpu): gfcc_dgemm_ozaki against exact integer / extended-precision
matrix products, and the whole sigma / solve path with option engine = 1 against the CPU oracle at the same tolerances as
the graded FP64 DMMA engine (1e-10 relative max-norm on sigma, 1e-8 on G; BASELINE.json north_star)."""
import numpy as np
import pytest
import torch

import gfcc_inputs as gi
import oracle
from gfcc_testutil import random_system, random_x, relmax

pytestmark = pytest.mark.gpu

TOL_SIGMA = 1e-10
TOL_G = 1e-8


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("M,N,K", [(128, 256, 128), (100, 200, 300), (1, 1, 1), (37, 5, 3), (300, 500, 1000), (777, 1111, 555)])
@pytest.mark.parametrize("ta", [0, 1])
@pytest.mark.parametrize("tb", [0, 1])
def test_ozaki_gemm_vs_extended_precision(M, N, K, ta, tb):
    """all four operand majors, ragged tails in M, N and K, alpha/beta; reference in 80-bit long double"""
    import paper_2010_04768_b200 as g
    rng = np.random.default_rng(M + 3 * N + 7 * K)
    A = rng.normal(size=(M, K)) * np.exp(rng.normal(size=(M, 1)))        # rows of different magnitude
    B = rng.normal(size=(K, N)) * np.exp(rng.normal(size=(1, N)))
    C0 = rng.normal(size=(M, N))
    Ad = dev(A.T).t() if ta else dev(A)
    Bd = dev(B.T).t() if tb else dev(B)
    Cd = dev(C0)
    g.gfcc_dgemm_ozaki(Ad, Bd, Cd, alpha=0.7, beta=-0.3, nslices=7)
    ref = (0.7 * (A.astype(np.longdouble) @ B.astype(np.longdouble)) - 0.3 * C0).astype(np.float64)
    # error bound of the scheme: per term 2^-49 x (row max of A) x (column max of B), K terms
    bound = K * 2.0 ** -46 * np.abs(A).max(axis=1)[:, None] * np.abs(B).max(axis=0)[None, :] + 1e-15 * np.abs(ref)
    assert (np.abs(Cd.cpu().numpy() - ref) <= bound).all()
    assert relmax(Cd.cpu().numpy(), ref) < 1e-12


def test_ozaki_gemm_exact_on_integers():
    """integer operands below 2^20 are represented exactly by 3 slices: the result must equal the integer product bit for bit"""
    import paper_2010_04768_b200 as g
    rng = np.random.default_rng(3)
    M, N, K = 260, 515, 1111
    A = rng.integers(-2 ** 19, 2 ** 19, size=(M, K)).astype(np.float64)
    B = rng.integers(-2 ** 19, 2 ** 19, size=(K, N)).astype(np.float64)
    ref = A.astype(np.int64) @ B.astype(np.int64)                          # |sum| < 1111 * 2^38 < 2^49: exact in int64
    C = g.gfcc_dgemm_ozaki(dev(A), dev(B), nslices=6).cpu().numpy()
    # |C| < 2^51: exactly representable; with 6 slices every digit product is kept (3 non-zero slices per operand)
    assert np.array_equal(C, ref.astype(np.float64))


def test_ozaki_gemm_slices_and_zero_rows():
    """accuracy follows 2^(-7 S); zero rows / columns and huge dynamic range between rows are handled by the per-row scale"""
    import paper_2010_04768_b200 as g
    rng = np.random.default_rng(11)
    M, N, K = 300, 260, 2000
    A = rng.normal(size=(M, K))
    B = rng.normal(size=(K, N))
    A[5] = 0.0
    B[:, 7] = 0.0
    A[9] *= 1e150
    A[11] *= 1e-150
    ref = (A.astype(np.longdouble) @ B.astype(np.longdouble)).astype(np.float64)
    rowscale = np.abs(ref).max(axis=1, keepdims=True) + 1e-300
    prev = None
    for S in (3, 5, 7, 8):
        C = g.gfcc_dgemm_ozaki(dev(A), dev(B), nslices=S).cpu().numpy()
        err = (np.abs(C - ref) / rowscale).max()
        assert err < 40 * 2.0 ** (-7 * S) * np.sqrt(K) + 4e-16, (S, err)
        assert (C[5] == 0).all() and (C[:, 7] == 0).all()
        if prev is not None:
            assert err < prev or err < 1e-15
        prev = err
    with pytest.raises(g.GfccError):
        g.gfcc_dgemm_ozaki(dev(A), dev(B), nslices=9)


@pytest.mark.parametrize("M,N,K", [(300, 520, 20000), (2560, 2560, 17000), (1000, 700, 140000)])
def test_ozaki_gemm_long_k_kernel(M, N, K):
    """K > 16384 selects the 128 x 256 read-modify-write kernel with the producer rendezvous (more tiles than SMs with a ragged
    last round, K long enough that one flush unit holds fewer pairs, ragged M/N/K).  Reference: 80-bit long-double dot products
    on the HOST for a sample of C entries (the four corners, the tile seams at 127/128 and 255/256, random interior entries)."""
    import paper_2010_04768_b200 as g
    rng = np.random.default_rng(M + N + K)
    A = rng.normal(size=(M, K))
    B = rng.normal(size=(K, N))
    C0 = rng.normal(size=(M, N))
    Ad, Bd = dev(A), dev(B)
    ms = np.concatenate([[0, M - 1, 127 % M, 128 % M], rng.integers(0, M, 60)])
    ns = np.concatenate([[0, N - 1, 255 % N, 256 % N], rng.integers(0, N, 60)])
    Al, Bl = A[ms].astype(np.longdouble), B[:, ns].astype(np.longdouble)
    prod = np.einsum("sk,ks->s", Al, Bl)                                    # exact to 2^-64 per term
    scale = np.sqrt(K) * 3.0                                                # typical |C| ~ sqrt(K)
    C = dev(C0)
    g.gfcc_dgemm_ozaki(Ad, Bd, C, alpha=-1.0, beta=1.0, nslices=7)
    got = C.cpu().numpy()[ms, ns]
    ref = (C0[ms, ns].astype(np.longdouble) - prod).astype(np.float64)
    assert np.abs(got - ref).max() / scale < 1e-12
    C = g.gfcc_dgemm_ozaki(Ad, Bd, nslices=7)
    got = C.cpu().numpy()[ms, ns]
    assert np.abs(got - prod.astype(np.float64)).max() / scale < 1e-12
    # a NaN / Inf in an operand row must reach the output row, not vanish in the slicing
    A[3, 17] = np.nan
    B[5, 2] = np.inf
    C = g.gfcc_dgemm_ozaki(dev(A), dev(B), nslices=7).cpu().numpy()
    assert np.isnan(C[3]).all() and not np.isfinite(C[:, 2]).any() and np.isfinite(C[4, 3])


def _make_pair(s):
    import paper_2010_04768_b200 as g
    orc = oracle.Oracle(s["o"], s["v"], s["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"], oracle.MODE_DEF)
    keep = [dev(s[k]) for k in ("fock", "T1", "T2p", "L1", "L2p", "Lchol")]
    h = g.gfcc_create(s["o"], s["v"], s["Q"], *keep)
    g.gfcc_set_option(h, "engine", 1)
    return g, orc, h


@pytest.mark.parametrize("o,v,Q,sym,nrhs", [(2, 2, 1, True, 1), (4, 6, 5, False, 2), (5, 7, 9, True, 4), (12, 37, 50, True, 5),
                                            (9, 130, 33, False, 7)])
def test_sigma_small_engine_ozaki(o, v, Q, sym, nrhs):
    s = random_system(o, v, Q, seed=7 + o + v, sym_L=sym, l_scale=0.3 if o < 9 else 0.1)
    g, orc, h = _make_pair(s)
    x1, x2 = random_x(o, v, nrhs, seed=5)
    w = -0.3 - 0.1 * np.arange(nrhs)
    S1, S2 = orc.sigma(w, 0.01, x1, x2)
    G1, G2 = g.gfcc_sigma_ip(h, w, 0.01, dev(x1), dev(x2))
    assert g.gfcc_get_stat(h, "oz_gemms") > 0 and g.gfcc_get_stat(h, "oz_fail") == 0
    assert relmax(G1.cpu().numpy(), S1) < TOL_SIGMA and relmax(G2.cpu().numpy(), S2) < TOL_SIGMA
    G2n = G2.cpu().numpy()
    assert np.array_equal(G2n, -G2n.transpose(0, 2, 1, 3))
    # small panels: several panels and a ragged last one go through the same code
    g.gfcc_set_option(h, "panel_bytes", 8.0 * o * v * v * 2)
    P1, P2 = g.gfcc_sigma_ip(h, w, 0.01, dev(x1), dev(x2))
    assert relmax(P2.cpu().numpy(), S2) < TOL_SIGMA
    # the two engines agree far below the parity tolerance
    g.gfcc_set_option(h, "engine", 0)
    D1, D2 = g.gfcc_sigma_ip(h, w, 0.01, dev(x1), dev(x2))
    assert relmax(G2n, D2.cpu().numpy()) < 1e-11
    g.gfcc_destroy(h)


def test_solve_small_engine_ozaki():
    o, v, Q = 6, 14, 24
    s = random_system(o, v, Q, seed=21, l_scale=0.1)
    g, orc, h = _make_pair(s)
    plist, ws = [o - 1, o - 2, o + 1], [-0.8, -0.4, -0.25]
    g.gfcc_set_option(h, "gmres_m", 300)
    G = g.gfcc_solve_ip(h, plist, ws, 0.01, 1e-11)
    Gd = orc.G_dense(plist, ws, 0.01)
    assert np.abs(G - Gd).max() < TOL_G * np.abs(Gd).max()
    assert g.gfcc_get_stat(h, "oz_fail") == 0
    g.gfcc_destroy(h)


@pytest.mark.parametrize("slices", [7, 6])
def test_config1_sigma_sampled_rows_engine_ozaki(slices):
    """config 1 at full size (o=40, v=160, Q=600, 64-RHS batch) on the INT8 engine against the row-sampled oracle; 7 digit
    slices is the default, 6 (21 instead of 28 digit products, ~1e-11 per GEMM) still meets the 1e-10 bar"""
    import paper_2010_04768_b200 as g
    cfg, nrhs, rsel = 1, 64, [0, 17, 63]
    c = gi.CONFIGS[cfg]
    o, v = c["o"], c["v"]
    s = gi.make_config(cfg, "cuda")
    host = {k: s[k].cpu().numpy() for k in ("fock", "T1", "T2p", "L1", "L2p", "Lchol")}
    h = g.gfcc_create(o, v, c["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"])
    g.gfcc_set_option(h, "ozaki_slices", slices)
    g.gfcc_set_option(h, "engine", 1)
    orc = oracle.Oracle(o, v, c["Q"], host["fock"], host["T1"], host["T2p"], host["L1"], host["L2p"], host["Lchol"], oracle.MODE_ROWS)
    X1, X2 = gi.trial_vectors(o, v, nrhs, gi.seed_of(cfg), "cuda")
    w = np.resize(np.linspace(c["wlo"], c["whi"], c["nw"]), nrhs)
    S1, S2 = g.gfcc_sigma_ip(h, w, c["eta"], X1, X2)
    torch.cuda.synchronize()
    assert g.gfcc_get_stat(h, "oz_fail") == 0
    rng = np.random.default_rng(101)
    trip = [(0, 1, 0), (0, o - 1, v - 1), (o - 2, o - 1, v // 2), (1, o // 2, 1)]
    while len(trip) < 12:
        i, j = sorted(rng.choice(o, 2, replace=False))
        trip.append((int(i), int(j), int(rng.integers(0, v))))
    trip = np.array(trip, dtype=np.int32)
    s1rows = [0, 7, 38, 39]
    R1, R2 = orc.sigma_rows(w[rsel], c["eta"], X1[rsel].cpu().numpy(), X2[rsel].cpu().numpy(), s1rows, trip)
    S1h, S2h = S1[rsel].cpu().numpy(), S2[rsel].cpu().numpy()
    e1 = np.abs(S1h[:, s1rows].T - R1).max() / float(S1.abs().max().item())
    e2 = np.abs(np.stack([S2h[:, i, j, a] for (i, j, a) in trip], axis=0) - R2).max() / float(S2.abs().max().item())
    g.gfcc_destroy(h)
    assert e1 < TOL_SIGMA and e2 < TOL_SIGMA, (e1, e2)
