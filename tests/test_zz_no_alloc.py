"""GPU test of the allocation-free entry point gfcc_dgemm_splitk_noalloc (include/gfcc.h): split-K FP64 GEMM whose partial sums
live in a file-scope static __device__ array of the library instead of a cudaMalloc'ed buffer.  Compared with the existing
GEMM path (gfcc_dgemm) at the tolerance of the GEMM unit tests (1e-13 relative max-norm), on calls in a row that share the
scratch (same shape, then a smaller and a differently split one, so that stale contents of the array would show).
This file is named to be collected LAST (the suite runs with pytest -x); it passes alone in a fresh process and after the others."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

TOL = 1e-13


def _rel(a, b):
    return float((a - b).abs().max() / b.abs().max())


def test_noalloc_splitk_gemm_matches_existing_path_on_consecutive_calls():
    import paper_2010_04768_b200 as g
    gen = torch.Generator(device="cuda").manual_seed(1234)
    rnd = lambda *s: torch.randn(s, dtype=torch.float64, device="cuda", generator=gen)
    # tall-skinny-K products (the shape class split-K is for): M x N small, K long and ragged
    cases = [(96, 40, 20011, 8, False, False), (96, 40, 20011, 8, False, False), (33, 130, 7777, 5, True, False),
             (128, 128, 4096, 16, False, True), (7, 3, 11, 64, False, False)]
    free_before = None
    for k, (M, N, K, S, ta, tb) in enumerate(cases):
        A = rnd(K, M).t() if ta else rnd(M, K)
        B = rnd(N, K).t() if tb else rnd(K, N)
        C0 = rnd(M, N)
        ref = g.gfcc_dgemm(A, B, C0.clone(), alpha=0.7, beta=-0.3)           # existing path: one pass over K, no scratch
        Cout = C0.clone()                                                    # torch's own allocation happens BEFORE the measurement
        torch.cuda.synchronize()
        if k == 1:
            free_before = torch.cuda.mem_get_info()[0]
        out = g.gfcc_dgemm_splitk_noalloc(A, B, Cout, alpha=0.7, beta=-0.3, splits=S)
        torch.cuda.synchronize()
        if k == 1:   # second call in a row, same kernels as the first: the device's free memory must not have moved
            assert torch.cuda.mem_get_info()[0] == free_before
        assert _rel(out, ref) < TOL, (k, _rel(out, ref))
        out2 = g.gfcc_dgemm_splitk_noalloc(A, B, torch.full((M, N), float("nan"), dtype=torch.float64, device="cuda"), splits=S)
        ref2 = g.gfcc_dgemm(A, B)
        assert _rel(out2, ref2) < TOL                                        # beta = 0 never reads C (NaN in, numbers out)
    # against an independent reference too (fp64 matmul on the host), so that a defect shared by both paths would show
    A, B = rnd(50, 3001), rnd(3001, 20)
    out = g.gfcc_dgemm_splitk_noalloc(A, B, torch.zeros((50, 20), dtype=torch.float64, device="cuda"), splits=7)
    assert _rel(out.cpu(), A.cpu() @ B.cpu()) < TOL


def test_noalloc_rejects_what_does_not_fit_the_builtin_scratch():
    import paper_2010_04768_b200 as g
    M = N = 1024                                       # 1 Mi doubles per part: 2 parts fit the 2 Mi-double scratch, 3 do not
    A = torch.ones((M, 64), dtype=torch.float64, device="cuda")
    B = torch.ones((64, N), dtype=torch.float64, device="cuda")
    C = torch.zeros((M, N), dtype=torch.float64, device="cuda")
    g.gfcc_dgemm_splitk_noalloc(A, B, C, splits=2)
    torch.cuda.synchronize()
    assert float(C.min()) == 64.0 and float(C.max()) == 64.0
    assert 2 * M * N == g.NOALLOC_SCRATCH_DOUBLES
    with pytest.raises(g.GfccError) as e:
        g.gfcc_dgemm_splitk_noalloc(A, B, C, splits=3)
    assert e.value.code == g.GFCC_EINVAL and "exceed the built-in scratch" in str(e.value)
    with pytest.raises(g.GfccError):
        g.gfcc_dgemm_splitk_noalloc(A, B, C, splits=0)
    # the failed calls launched nothing and left C alone; the next valid call works
    g.gfcc_dgemm_splitk_noalloc(A, B, C, alpha=2.0, splits=1)
    torch.cuda.synchronize()
    assert float(C.min()) == 128.0
