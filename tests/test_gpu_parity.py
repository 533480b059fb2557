"""GPU parity tests (run with -m gpu on a B200): the CUDA path vs the CPU oracle, element by element, through the
C ABI.  Tolerances are BASELINE.json north_star's: 1e-10 relative max-norm on sigma, 1e-8 relative on G_pq."""
import numpy as np
import pytest
import torch

import oracle
from gfcc_testutil import random_system, random_x, relmax, to_numpy_system

pytestmark = pytest.mark.gpu

TOL_SIGMA = 1e-10
TOL_G = 1e-8


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


def make_pair(s, mode=oracle.MODE_DEF):
    import paper_2010_04768_b200 as g
    orc = oracle.Oracle(s["o"], s["v"], s["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"], mode)
    keep = [dev(s[k]) for k in ("fock", "T1", "T2p", "L1", "L2p", "Lchol")]
    h = g.gfcc_create(s["o"], s["v"], s["Q"], *keep)
    return g, orc, h


# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("M,N,K", [(128, 128, 16), (200, 300, 77), (1, 512, 100), (660, 96, 33), (37, 5, 3), (777, 1111, 555)])
@pytest.mark.parametrize("ta", [0, 1])
@pytest.mark.parametrize("tb", [0, 1])
def test_dmma_gemm_engine(M, N, K, ta, tb):
    """unit test of the FP64 tensor-core GEMM against a plain fp64 matmul (all four operand majors, ragged tails)"""
    import paper_2010_04768_b200 as g
    rng = np.random.default_rng(M + 3 * N + 7 * K)
    A = rng.normal(size=(M, K))
    B = rng.normal(size=(K, N))
    C0 = rng.normal(size=(M, N))
    Ad = dev(A.T).t() if ta else dev(A)
    Bd = dev(B.T).t() if tb else dev(B)
    Cd = dev(C0)
    g.gfcc_dgemm(Ad, Bd, Cd, alpha=0.7, beta=-0.3)
    ref = 0.7 * (A @ B) - 0.3 * C0
    assert relmax(Cd.cpu().numpy(), ref) < 1e-13
    Cd = g.gfcc_dgemm(Ad, Bd)
    assert relmax(Cd.cpu().numpy(), A @ B) < 1e-13


def check_intermediates(g, orc, h, s):
    o, v = s["o"], s["v"]
    iu = np.triu_indices(o, 1)
    for name in ("Fme", "Fmi", "Fae"):
        ref = orc.get(name)
        assert relmax(g.gfcc_get_intermediate(h, name).cpu().numpy().reshape(ref.shape), ref) < 1e-12, name
    W = orc.get("Wmnij")
    ref = W[iu[0], iu[1]][:, iu[0], iu[1]].T                         # [(i<j)][(m<n)]
    assert relmax(g.gfcc_get_intermediate(h, "Wmnij").cpu().numpy().reshape(ref.shape), ref) < 1e-12
    Wm = orc.get("Wmbij")
    ref = np.transpose(Wm[:, :, iu[1], iu[0]], (2, 1, 0))            # [pair][b][m] = W[m,b,j,i]
    assert relmax(g.gfcc_get_intermediate(h, "Wmbij").cpu().numpy().reshape(ref.shape), ref) < 1e-12


@pytest.mark.parametrize("o,v,Q,sym,nrhs", [(2, 2, 1, True, 1), (3, 3, 4, True, 3), (4, 6, 5, False, 2), (5, 7, 9, True, 4),
                                            (12, 37, 50, True, 5), (9, 130, 33, False, 7)])
def test_create_and_sigma_small(o, v, Q, sym, nrhs):
    s = random_system(o, v, Q, seed=7 + o + v, sym_L=sym, l_scale=0.3 if o < 9 else 0.1)
    g, orc, h = make_pair(s)
    check_intermediates(g, orc, h, s)
    x1, x2 = random_x(o, v, nrhs, seed=5)
    w = -0.3 - 0.1 * np.arange(nrhs)
    S1, S2 = orc.sigma(w, 0.01, x1, x2)
    G1, G2 = g.gfcc_sigma_ip(h, w, 0.01, dev(x1), dev(x2))
    assert relmax(G1.cpu().numpy(), S1) < TOL_SIGMA and relmax(G2.cpu().numpy(), S2) < TOL_SIGMA
    # bit-level structure: antisymmetric, zero diagonal
    G2n = G2.cpu().numpy()
    assert np.array_equal(G2n, -G2n.transpose(0, 2, 1, 3))
    # host-buffer entry point gives the same bits
    H1, H2 = g.gfcc_sigma_ip_host(h, w, 0.01, x1, x2)
    assert np.array_equal(H1, G1.cpu().numpy()) and np.array_equal(H2, G2n)
    # ... also into caller-provided (pinned) host outputs
    P1 = torch.empty(x1.shape, dtype=torch.complex128, pin_memory=True)
    P2 = torch.empty(x2.shape, dtype=torch.complex128, pin_memory=True)
    g.gfcc_sigma_ip_host(h, w, 0.01, x1, x2, out=(P1, P2))
    assert np.array_equal(P1.numpy(), H1) and np.array_equal(P2.numpy(), H2)
    with pytest.raises(g.GfccError):
        g.gfcc_sigma_ip_host(h, w, 0.01, x1, x2, out=(P2, P1))
    # exact shift identity on the GPU path too
    T1, T2 = g.gfcc_sigma_ip(h, w + 0.25, 0.01, dev(x1), dev(x2))
    assert relmax((T2 - G2).cpu().numpy(), 0.25 * x2) < 1e-12
    g.gfcc_destroy(h)


@pytest.mark.parametrize("o,v,Q,sym", [(3, 3, 4, True), (4, 6, 5, False), (6, 11, 12, True)])
def test_solve_small_vs_dense_lu(o, v, Q, sym):
    s = random_system(o, v, Q, seed=17 + o, sym_L=sym, l_scale=0.2)
    g, orc, h = make_pair(s)
    plist = [o - 1, 0, o + 1, o + v - 1]          # occupied and virtual targets
    ws = [-0.4, -0.9, -0.15]
    Gd = orc.G_dense(plist, ws, 0.02)
    g.gfcc_set_option(h, "gmres_m", 500)
    G, X1, X2 = g.gfcc_solve_ip(h, plist, ws, 0.02, 1e-11, return_x=True)
    assert relmax(G, Gd) < TOL_G
    # solver-independent check: plug the GPU's X into the ORACLE sigma, true residual <= tol
    X1n, X2n = X1.cpu().numpy(), X2.cpu().numpy()
    wr = np.array([ws[iw] for ip in range(len(plist)) for iw in range(len(ws))])
    S1, S2 = orc.sigma(wr, 0.02, X1n, X2n)
    for r in range(len(wr)):
        b1, b2 = orc.rhs(plist[r // len(ws)])
        res = orc.pack(b1 - S1[r], b2 - S2[r])
        assert np.linalg.norm(res) / np.linalg.norm(orc.pack(b1, b2)) < 1e-9
    # restarted GMRES, zero initial guess, small batches: same G
    g.gfcc_set_option(h, "gmres_m", 30)     # restarted (n = 12 / 40 / 171 unknowns); GMRES(m) may stagnate for tiny m
    g.gfcc_set_option(h, "x0", 0)
    g.gfcc_set_option(h, "max_batch", 5)
    g.gfcc_set_option(h, "gmres_maxit", 20000)
    G2 = g.gfcc_solve_ip(h, plist, ws, 0.02, 1e-11)
    assert relmax(G2, Gd) < TOL_G
    rel, its = g.gfcc_get_residuals(h, len(wr))
    assert (rel <= 1e-11).all() and (its > 0).all()
    g.gfcc_destroy(h)


def test_error_paths():
    import paper_2010_04768_b200 as g
    s = random_system(3, 3, 2, seed=1)
    g_, orc, h = make_pair(s)
    with pytest.raises(g.GfccError) as e:
        g.gfcc_solve_ip(h, [99], [-0.5], 0.01, 1e-8)
    assert e.value.code == g.GFCC_EINVAL
    with pytest.raises(g.GfccError):
        g.gfcc_set_option(h, "no_such_option", 1)
    g.gfcc_set_option(h, "gmres_maxit", 2)
    with pytest.raises(g.GfccError) as e:
        g.gfcc_solve_ip(h, [2], [-0.5], 0.01, 1e-13)
    assert e.value.code == g.GFCC_ENOCONV
    g.gfcc_destroy(h)


# ---------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def cfg0():
    import gfcc_inputs
    s = to_numpy_system(gfcc_inputs.make_config(0, "cpu"))
    g, orc, h = make_pair(s)
    yield s, g, orc, h
    g.gfcc_destroy(h)


def test_config0_sigma(cfg0):
    import gfcc_inputs
    s, g, orc, h = cfg0
    check_intermediates(g, orc, h, s)
    nrhs = 32
    X1, X2 = gfcc_inputs.trial_vectors(8, 24, nrhs, gfcc_inputs.seed_of(0))
    w = np.repeat(np.asarray(s["omegas"]), 4)
    S1, S2 = orc.sigma(w, s["eta"], X1.numpy(), X2.numpy())
    G1, G2 = g.gfcc_sigma_ip(h, w, s["eta"], X1.cuda(), X2.cuda())
    assert relmax(G1.cpu().numpy(), S1) < TOL_SIGMA and relmax(G2.cpu().numpy(), S2) < TOL_SIGMA


def test_config0_solve(cfg0):
    s, g, orc, h = cfg0
    ws = np.asarray(s["omegas"])
    Gd = orc.G_dense(s["targets"], ws, s["eta"])
    g.gfcc_set_option(h, "gmres_m", 400)
    G = g.gfcc_solve_ip(h, s["targets"], ws, s["eta"], 1e-11)
    assert G.shape == (8, 4, 4)
    for iw in range(len(ws)):
        assert np.abs(G[iw] - Gd[iw]).max() <= TOL_G * np.abs(Gd[iw]).max()
    # the config's own tolerance with the default restart length policy also meets the G tolerance
    g.gfcc_set_option(h, "gmres_m", 300)
    G = g.gfcc_solve_ip(h, s["targets"], ws, s["eta"], s["tol"])
    assert relmax(G, Gd) < TOL_G
    # fixed-iteration mode: the k-step GMRES iterate is unique (reading 19) -> compare X with the oracle's
    g.gfcc_set_option(h, "gmres_fixed", 25)
    Gf, X1, X2 = g.gfcc_solve_ip(h, s["targets"][:1], ws[:2], s["eta"], 1e-30, return_x=True)
    g.gfcc_set_option(h, "gmres_fixed", 0)
    for iw in range(2):
        # 25 Arnoldi steps + 1 residual evaluation = 26 sigma applications in the oracle's counting
        x1, x2, nit, rr = orc.gmres(s["targets"][0], ws[iw], s["eta"], 1e-30, m=25, maxit=26, x0kind=1)
        assert relmax(orc.pack(X1[iw].cpu().numpy(), X2[iw].cpu().numpy()), orc.pack(x1, x2)) < 1e-8


def test_failed_workspace_allocation_leaves_the_handle_usable():
    """a workspace allocation that fails half-way (device memory nearly full) must return GFCC_ENOMEM and leave the
    handle clean, so that the same call succeeds once memory is available again (no launch on half-allocated buffers)."""
    import gc
    s = random_system(12, 37, 50, seed=3, l_scale=0.1)
    g, orc, h = make_pair(s)
    o, v = 12, 37
    x1, x2 = random_x(o, v, 4, seed=11)
    w4 = np.array([-0.3, -0.5, 0.2, -0.9])
    ref1, ref2 = g.gfcc_sigma_ip(h, w4, 0.01, dev(x1), dev(x2))            # loads the kernels, small workspace
    torch.cuda.synchronize()
    nrhs = 2048                                                            # workspace of this batch: 3 x 175 MB + vectors
    X1 = dev(np.tile(x1, (nrhs // 4, 1)))
    X2 = dev(np.tile(x2, (nrhs // 4, 1, 1, 1)))
    S1 = torch.empty_like(X1)
    S2 = torch.empty_like(X2)
    wbig = np.tile(w4, nrhs // 4)
    gc.collect()
    torch.cuda.empty_cache()
    free = torch.cuda.mem_get_info()[0]
    hog = torch.empty(free - 300 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # leave ~300 MB: the 2nd/3rd buffer cannot fit
    with pytest.raises(g.GfccError) as e:
        g.gfcc_sigma_ip(h, wbig, 0.01, X1, X2, S1, S2)
    assert e.value.code == g.GFCC_ENOMEM
    with pytest.raises(g.GfccError) as e:                                   # again, same batch width: still an error, not a crash
        g.gfcc_sigma_ip(h, wbig, 0.01, X1, X2, S1, S2)
    assert e.value.code == g.GFCC_ENOMEM
    del hog
    torch.cuda.empty_cache()
    g.gfcc_sigma_ip(h, wbig, 0.01, X1, X2, S1, S2)                          # memory is back: the same call works
    torch.cuda.synchronize()
    assert relmax(S1[:4].cpu().numpy(), ref1.cpu().numpy()) < 1e-13 and relmax(S2[-4:].cpu().numpy(), ref2.cpu().numpy()) < 1e-13
    G1, G2 = g.gfcc_sigma_ip(h, w4, 0.01, dev(x1), dev(x2))                 # and the small batch still does
    assert relmax(G2.cpu().numpy(), ref2.cpu().numpy()) < 1e-13
    g.gfcc_destroy(h)
