"""Thin Python binding of libgfcc_b200.so (include/gfcc.h) -- argument marshalling only.

Every step of the GFCCSD-IP hot path (Eq. 5, Eq. 7-8) runs in
the hand-written CUDA kernels of the library; PyTorch is used for device memory and streams only.
There is no CPU fallback: importing works without a GPU (so that the symbol table can be checked), but every
compute call needs a CUDA device and raises GfccError otherwise.  The CPU oracle (oracle/) is never imported
here.

Functions have the names of the C entry points and take torch CUDA tensors (float64 / complex128):
    h = gfcc_create(o, v, Q, fock, T1, T2, L1, L2, Lchol)
    S1, S2 = gfcc_sigma_ip(h, omega, eta, X1, X2)
    G = gfcc_solve_ip(h, p, omega, eta, tol)
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgfcc_b200.so")

GFCC_OK, GFCC_EINVAL, GFCC_ENOMEM, GFCC_ECUDA, GFCC_ENOCONV = 0, -1, -2, -3, -4

EXPORTS = ["gfcc_create", "gfcc_create_closed_shell", "gfcc_sigma_ip", "gfcc_sigma_ip_host", "gfcc_solve_ip", "gfcc_solve_ip_x", "gfcc_set_stream",
           "gfcc_set_option", "gfcc_get_stat", "gfcc_get_residuals", "gfcc_get_residual_history", "gfcc_assemble_g",
           "gfcc_get_intermediate", "gfcc_last_error",
           "gfcc_destroy", "gfcc_dgemm", "gfcc_dgemm_splitk_noalloc", "gfcc_dgemm_ozaki", "gfcc_probe_fp64_peak", "gfcc_mor_reset", "gfcc_mor_extend", "gfcc_mor_solve",
           "gfcc_mor_get", "gfcc_spectral_adaptive", "gfcc_sigma_ea", "gfcc_solve_ea", "gfcc_solve_ea_x", "gfcc_assemble_g_ea"]


class GfccError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"gfcc error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load the CUDA library; fails loudly if it has not been built (python -m paper_2010_04768_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise GfccError(GFCC_ECUDA, f"{LIB_PATH} is missing: build it with `python -m paper_2010_04768_b200.build` "
                                    "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, dp, ip = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
    ci, cd, cll = ctypes.c_int, ctypes.c_double, ctypes.c_longlong
    L.gfcc_create.argtypes = [ci, ci, ci, vp, vp, vp, vp, vp, vp, ctypes.POINTER(vp)]
    L.gfcc_create_closed_shell.argtypes = [ci, ci, ci, vp, vp, vp, vp, vp, vp, ctypes.POINTER(vp)]
    L.gfcc_sigma_ip.argtypes = [vp, ci, dp, cd, vp, vp, vp, vp]
    L.gfcc_sigma_ip_host.argtypes = [vp, ci, dp, cd, vp, vp, vp, vp]
    L.gfcc_solve_ip.argtypes = [vp, ci, ip, ci, dp, cd, cd, vp]
    L.gfcc_solve_ip_x.argtypes = [vp, ci, ip, ci, dp, cd, cd, vp, vp, vp]
    L.gfcc_set_stream.argtypes = [vp, vp]
    L.gfcc_set_option.argtypes = [vp, ctypes.c_char_p, cd]
    L.gfcc_get_stat.argtypes = [vp, ctypes.c_char_p, dp]
    L.gfcc_get_residuals.argtypes = [vp, ci, dp, ip]
    L.gfcc_get_residual_history.argtypes = [vp, ci, ci, dp, ip]
    L.gfcc_assemble_g.argtypes = [vp, ci, vp, vp, ci, ip, vp]
    L.gfcc_get_intermediate.argtypes = [vp, ctypes.c_char_p, vp]
    L.gfcc_sigma_ea.argtypes = [vp, ci, dp, cd, vp, vp, vp, vp]
    L.gfcc_solve_ea.argtypes = [vp, ci, ip, ci, dp, cd, cd, vp]
    L.gfcc_solve_ea_x.argtypes = [vp, ci, ip, ci, dp, cd, cd, vp, vp, vp]
    L.gfcc_assemble_g_ea.argtypes = [vp, ci, vp, vp, ci, ip, vp]
    L.gfcc_get_intermediate.restype = cll
    L.gfcc_last_error.argtypes = [vp]
    L.gfcc_last_error.restype = ctypes.c_char_p
    L.gfcc_destroy.argtypes = [vp]
    L.gfcc_dgemm.argtypes = [vp, ci, ci, ci, cd, vp, cll, cll, vp, cll, cll, cd, vp, cll, cll]
    L.gfcc_dgemm_splitk_noalloc.argtypes = [vp, ci, ci, ci, cd, vp, cll, cll, vp, cll, cll, cd, vp, cll, cll, ci]
    L.gfcc_dgemm_ozaki.argtypes = [vp, ci, ci, ci, cd, vp, cll, cll, vp, cll, cll, cd, vp, cll, cll, ci, dp, dp]
    L.gfcc_probe_fp64_peak.argtypes = [vp, ci, ci, dp]
    L.gfcc_mor_reset.argtypes = [vp, ci]
    L.gfcc_mor_extend.argtypes = [vp, ci, vp, vp, cd, ip]
    L.gfcc_mor_solve.argtypes = [vp, ci, ip, ci, dp, cd, vp, dp]
    L.gfcc_mor_get.argtypes = [vp, ctypes.c_char_p, vp]
    L.gfcc_mor_get.restype = cll
    L.gfcc_spectral_adaptive.argtypes = [vp, ci, ip, cd, cd, cd, cd, cd, cd, ci, cd, ci, dp, vp, ip, ip, ip]
    for name in EXPORTS:
        if name not in ("gfcc_get_intermediate", "gfcc_last_error", "gfcc_mor_get"):
            getattr(L, name).restype = ci
    _lib = L
    return L


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise GfccError(GFCC_ECUDA, "no CUDA device: the GFCC hot path has no CPU fallback")
    return torch


def _dev(t, dtype):
    torch = _torch()
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise GfccError(GFCC_EINVAL, f"expected a contiguous CUDA tensor of {dtype}")
    return ctypes.c_void_p(t.data_ptr())


def _check(h, rc, allow=()):
    if rc != GFCC_OK and rc not in allow:
        msg = lib().gfcc_last_error(h.ptr if h is not None else None)
        raise GfccError(rc, msg.decode() if msg else "")
    return rc


class Handle:
    """Opaque gfcc_handle plus references that keep the BORROWED tensors (T2, L2) alive."""

    def __init__(self, ptr, o, v, Q, keep):
        self.ptr, self.o, self.v, self.Q, self._keep = ptr, o, v, Q, keep

    def __del__(self):
        try:
            gfcc_destroy(self)
        except Exception:
            pass


def gfcc_create(o, v, Q, fock, T1, T2, L1, L2, Lchol, stream=None):
    torch = _torch()
    f64 = torch.float64
    N, npair, ntri = o + v, o * (o - 1) // 2, v * (v - 1) // 2
    for t, n, name in ((fock, N * N, "fock"), (T1, o * v, "T1"), (T2, npair * v * v, "T2"), (L1, o * v, "L1"),
                       (L2, npair * ntri, "L2"), (Lchol, Q * N * N, "Lchol")):
        if t.numel() != n:
            raise GfccError(GFCC_EINVAL, f"{name} has {t.numel()} elements, expected {n}")
    out = ctypes.c_void_p()
    rc = lib().gfcc_create(o, v, Q, _dev(fock, f64), _dev(T1, f64), _dev(T2, f64), _dev(L1, f64), _dev(L2, f64),
                           _dev(Lchol, f64), ctypes.byref(out))
    _check(None, rc)
    h = Handle(out, o, v, Q, (T2, L2))
    if stream is not None:
        gfcc_set_stream(h, stream)
    return h


def gfcc_create_closed_shell(no, nv, Q, fock, T1, T2, L1, L2, Lchol, stream=None):
    """closed-shell (spin-restricted) spatial tensors -> spin-orbital handle with o = 2 no, v = 2 nv (include/gfcc.h).
    spin_orbital(p, alpha) = p for p < no, 2 no + (p - no) otherwise."""
    torch = _torch()
    f64 = torch.float64
    Ns = no + nv
    for t, n, name in ((fock, Ns * Ns, "fock"), (T1, no * nv, "T1"), (T2, no * no * nv * nv, "T2"), (L1, no * nv, "L1"),
                       (L2, no * no * nv * nv, "L2"), (Lchol, Q * Ns * Ns, "Lchol")):
        if t.numel() != n:
            raise GfccError(GFCC_EINVAL, f"{name} has {t.numel()} elements, expected {n}")
    out = ctypes.c_void_p()
    rc = lib().gfcc_create_closed_shell(no, nv, Q, _dev(fock, f64), _dev(T1, f64), _dev(T2, f64), _dev(L1, f64), _dev(L2, f64),
                                        _dev(Lchol, f64), ctypes.byref(out))
    _check(None, rc)
    h = Handle(out, 2 * no, 2 * nv, Q, None)
    if stream is not None:
        gfcc_set_stream(h, stream)
    return h


def gfcc_destroy(h):
    if h.ptr:
        lib().gfcc_destroy(h.ptr)
        h.ptr = None
        h._keep = None


def gfcc_set_stream(h, stream):
    """stream: torch.cuda.Stream or a raw cudaStream_t integer."""
    raw = getattr(stream, "cuda_stream", stream)
    _check(h, lib().gfcc_set_stream(h.ptr, ctypes.c_void_p(raw)))


def gfcc_set_option(h, key, val):
    _check(h, lib().gfcc_set_option(h.ptr, key.encode(), float(val)))


def gfcc_get_stat(h, key):
    out = ctypes.c_double()
    _check(h, lib().gfcc_get_stat(h.ptr, key.encode(), ctypes.byref(out)))
    return out.value


def gfcc_get_residuals(h, n):
    rel = np.empty(n, dtype=np.float64)
    its = np.empty(n, dtype=np.int32)
    _check(h, lib().gfcc_get_residuals(h.ptr, n, rel.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                       its.ctypes.data_as(ctypes.POINTER(ctypes.c_int))))
    return rel, its


def gfcc_get_residual_history(h, rhs):
    """relative residual of right-hand side `rhs` of the last solve after each of its sigma applications (numpy array)."""
    n = ctypes.c_int(0)
    _check(h, lib().gfcc_get_residual_history(h.ptr, int(rhs), 0, None, ctypes.byref(n)))
    out = np.empty(n.value, dtype=np.float64)
    if n.value:
        _check(h, lib().gfcc_get_residual_history(h.ptr, int(rhs), n.value, out.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                                  ctypes.byref(n)))
    return out


def gfcc_assemble_g(h, X1, X2, q):
    """G assembly alone: X1 [nrhs,o], X2 [nrhs,o,o,v] complex128 CUDA tensors, q host ints -> G [nrhs, nq] numpy complex128."""
    torch = _torch()
    qa = np.ascontiguousarray(q, dtype=np.int32)
    nrhs = X1.shape[0]
    if X1.numel() != nrhs * h.o or X2.numel() != nrhs * h.o * h.o * h.v:
        raise GfccError(GFCC_EINVAL, "X1/X2 shape mismatch")
    G = np.empty((nrhs, len(qa)), dtype=np.complex128)
    _check(h, lib().gfcc_assemble_g(h.ptr, nrhs, _dev(X1, torch.complex128), _dev(X2, torch.complex128), len(qa),
                                    qa.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), G.ctypes.data))
    return G


def gfcc_get_intermediate(h, name):
    torch = _torch()
    n = lib().gfcc_get_intermediate(h.ptr, name.encode(), None)
    if n < 0:
        _check(h, int(n))
    out = torch.empty(int(n), dtype=torch.float64, device="cuda")
    n2 = lib().gfcc_get_intermediate(h.ptr, name.encode(), ctypes.c_void_p(out.data_ptr()))
    if n2 < 0:
        _check(h, int(n2))
    return out


def _omega(omega, n):
    om = np.ascontiguousarray(np.broadcast_to(np.asarray(omega, dtype=np.float64), (n,)))
    return om, om.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def gfcc_sigma_ip(h, omega, eta, X1, X2, S1=None, S2=None):
    """X1 [nrhs,o], X2 [nrhs,o,o,v] complex128 CUDA tensors -> (S1, S2). Asynchronous on the handle's stream."""
    torch = _torch()
    c128 = torch.complex128
    nrhs = X1.shape[0]
    if X1.numel() != nrhs * h.o or X2.numel() != nrhs * h.o * h.o * h.v:
        raise GfccError(GFCC_EINVAL, "X1/X2 shape mismatch")
    if S1 is None:
        S1 = torch.empty_like(X1)
    if S2 is None:
        S2 = torch.empty_like(X2)
    om, omp = _omega(omega, nrhs)
    _check(h, lib().gfcc_sigma_ip(h.ptr, nrhs, omp, float(eta), _dev(X1, c128), _dev(X2, c128), _dev(S1, c128), _dev(S2, c128)))
    return S1, S2


def gfcc_sigma_ip_host(h, omega, eta, X1, X2, out=None):
    """Same with HOST numpy complex128 arrays (or pinned CPU tensors); copies are inside the call.  out = (S1, S2): optional
    preallocated host outputs of the same shapes (e.g. views of pinned tensors: the device-to-host copy then runs at full speed)."""
    X1 = np.ascontiguousarray(X1.numpy() if hasattr(X1, "numpy") else X1, dtype=np.complex128)
    X2 = np.ascontiguousarray(X2.numpy() if hasattr(X2, "numpy") else X2, dtype=np.complex128)
    nrhs = X1.shape[0]
    if out is not None:
        S1, S2 = (t.numpy() if hasattr(t, "numpy") else t for t in out)
        if (S1.shape != X1.shape or S2.shape != X2.shape or S1.dtype != np.complex128 or S2.dtype != np.complex128
                or not S1.flags.c_contiguous or not S2.flags.c_contiguous):
            raise GfccError(GFCC_EINVAL, "gfcc_sigma_ip_host: out must be contiguous complex128 arrays shaped like X1, X2")
    else:
        S1 = np.empty_like(X1)
        S2 = np.empty_like(X2)
    om, omp = _omega(omega, nrhs)
    _check(h, lib().gfcc_sigma_ip_host(h.ptr, nrhs, omp, float(eta), X1.ctypes.data, X2.ctypes.data, S1.ctypes.data, S2.ctypes.data))
    return S1, S2


def gfcc_solve_ip(h, p, omega, eta, tol, return_x=False, allow_noconv=False):
    """p: target spin-orbitals (host ints), omega: host floats -> G [nw, np, np] complex128 numpy array (host).
    return_x: also return device tensors X1 [np*nw, o], X2 [np*nw, o, o, v] (RHS order r = ip*nw + iw)."""
    torch = _torch()
    pa = np.ascontiguousarray(p, dtype=np.int32)
    npn, nw = len(pa), len(np.atleast_1d(omega))
    om, omp = _omega(np.atleast_1d(omega), nw)
    G = np.empty((nw, npn, npn), dtype=np.complex128)
    allow = (GFCC_ENOCONV,) if allow_noconv else ()
    if return_x:
        X1 = torch.empty((npn * nw, h.o), dtype=torch.complex128, device="cuda")
        X2 = torch.empty((npn * nw, h.o, h.o, h.v), dtype=torch.complex128, device="cuda")
        rc = lib().gfcc_solve_ip_x(h.ptr, npn, pa.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), nw, omp, float(eta), float(tol),
                                   G.ctypes.data, ctypes.c_void_p(X1.data_ptr()), ctypes.c_void_p(X2.data_ptr()))
        _check(h, rc, allow)
        return G, X1, X2
    rc = lib().gfcc_solve_ip(h.ptr, npn, pa.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), nw, omp, float(eta), float(tol),
                             G.ctypes.data)
    _check(h, rc, allow)
    return G


def gfcc_spectral_adaptive(h, p, wmin, wmax, dw, eta, tol, spec_tol=1e-3, max_levels=0, droptol=1e-8, allow_noconv=False):
    """Alg. 1 level loop with adaptive midpoint refinement (include/gfcc.h).  Returns dict(w, A, G, level_of, levels, m)."""
    _torch()
    pa = np.ascontiguousarray(p, dtype=np.int32)
    n = int(round((wmax - wmin) / dw)) + 1 if dw > 0 else 0
    n = max(n, 1)                                  # the library rejects an empty window or a grid of fewer than 3 points
    A = np.zeros(n, dtype=np.float64)
    G = np.zeros((n, len(pa), len(pa)), dtype=np.complex128)
    lev = np.zeros(n, dtype=np.int32)
    levels, m = ctypes.c_int(), ctypes.c_int()
    rc = lib().gfcc_spectral_adaptive(h.ptr, len(pa), pa.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), float(wmin), float(wmax),
                                      float(dw), float(eta), float(tol), float(spec_tol), int(max_levels), float(droptol), n,
                                      A.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), G.ctypes.data,
                                      lev.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), ctypes.byref(levels), ctypes.byref(m))
    _check(h, rc, (GFCC_ENOCONV,) if allow_noconv else ())
    return {"w": wmin + dw * np.arange(n), "A": A, "G": G, "level_of": lev, "levels": levels.value, "m": m.value}


def gfcc_dgemm(A, B, C=None, alpha=1.0, beta=0.0, stream=0):
    """C = alpha * A @ B + beta * C through the DMMA engine; A, B, C are 2-D float64 CUDA tensors (any strides with one
    unit stride per operand)."""
    torch = _torch()
    M, K = A.shape
    K2, N = B.shape
    assert K == K2
    if C is None:
        C = torch.zeros((M, N), dtype=torch.float64, device=A.device)
    rc = lib().gfcc_dgemm(ctypes.c_void_p(stream), M, N, K, float(alpha), ctypes.c_void_p(A.data_ptr()), A.stride(0), A.stride(1),
                          ctypes.c_void_p(B.data_ptr()), B.stride(0), B.stride(1), float(beta), ctypes.c_void_p(C.data_ptr()),
                          C.stride(0), C.stride(1))
    if rc != GFCC_OK:
        raise GfccError(rc, "gfcc_dgemm failed")
    return C


NOALLOC_SCRATCH_DOUBLES = 1 << 21


def gfcc_dgemm_splitk_noalloc(A, B, C, alpha=1.0, beta=0.0, splits=8, stream=0):
    """C = alpha * A @ B + beta * C, split-K, with the partial sums in the library's built-in static device scratch: the call allocates
    nothing (C must be given).  Raises GfccError(GFCC_EINVAL) when parts * M * N exceeds NOALLOC_SCRATCH_DOUBLES."""
    _torch()
    M, K = A.shape
    K2, N = B.shape
    assert K == K2 and tuple(C.shape) == (M, N)
    raw = getattr(stream, "cuda_stream", stream)
    rc = lib().gfcc_dgemm_splitk_noalloc(ctypes.c_void_p(raw), M, N, K, float(alpha), ctypes.c_void_p(A.data_ptr()), A.stride(0),
                                         A.stride(1), ctypes.c_void_p(B.data_ptr()), B.stride(0), B.stride(1), float(beta),
                                         ctypes.c_void_p(C.data_ptr()), C.stride(0), C.stride(1), int(splits))
    if rc != GFCC_OK:
        msg = lib().gfcc_last_error(None)
        raise GfccError(rc, msg.decode() if msg else "gfcc_dgemm_splitk_noalloc failed")
    return C


def gfcc_dgemm_ozaki(A, B, C=None, alpha=1.0, beta=0.0, nslices=7, stream=0, return_times=False):
    """C = alpha * A @ B + beta * C on the INT8 tensor pipe with FP64 accuracy (error-free slicing; include/gfcc.h)."""
    torch = _torch()
    M, K = A.shape
    K2, N = B.shape
    assert K == K2
    if C is None:
        C = torch.zeros((M, N), dtype=torch.float64, device=A.device)
    ms_s, ms_g = ctypes.c_double(), ctypes.c_double()
    rc = lib().gfcc_dgemm_ozaki(ctypes.c_void_p(stream), M, N, K, float(alpha), ctypes.c_void_p(A.data_ptr()), A.stride(0),
                                A.stride(1), ctypes.c_void_p(B.data_ptr()), B.stride(0), B.stride(1), float(beta),
                                ctypes.c_void_p(C.data_ptr()), C.stride(0), C.stride(1), int(nslices), ctypes.byref(ms_s),
                                ctypes.byref(ms_g))
    if rc != GFCC_OK:
        raise GfccError(rc, "gfcc_dgemm_ozaki failed")
    return (C, ms_s.value, ms_g.value) if return_times else C


def gfcc_probe_fp64_peak(iters=20000, reps=5, stream=0):
    """Measured FP64 DMMA issue-rate ceiling of this GPU in TFLOP/s (roofline denominator of the sigma GEMMs)."""
    _torch()
    out = ctypes.c_double()
    raw = getattr(stream, "cuda_stream", stream)
    rc = lib().gfcc_probe_fp64_peak(ctypes.c_void_p(raw), int(iters), int(reps), ctypes.byref(out))
    if rc != GFCC_OK:
        raise GfccError(rc, "gfcc_probe_fp64_peak failed")
    return out.value


# ---- EA / advanced part (Eq. 6; second terms of Eq. 7-8) ------------------------------------------
def gfcc_sigma_ea(h, omega, eta, Y1, Y2, S1=None, S2=None):
    """Y1 [nrhs,v], Y2 [nrhs,o,v,v] complex128 CUDA tensors -> (S1, S2) = (omega + i eta) Y - Hbar Y."""
    torch = _torch()
    c128 = torch.complex128
    nrhs = Y1.shape[0]
    if Y1.numel() != nrhs * h.v or Y2.numel() != nrhs * h.o * h.v * h.v:
        raise GfccError(GFCC_EINVAL, "Y1/Y2 shape mismatch")
    if S1 is None:
        S1 = torch.empty_like(Y1)
    if S2 is None:
        S2 = torch.empty_like(Y2)
    om, omp = _omega(omega, nrhs)
    _check(h, lib().gfcc_sigma_ea(h.ptr, nrhs, omp, float(eta), _dev(Y1, c128), _dev(Y2, c128), _dev(S1, c128), _dev(S2, c128)))
    return S1, S2


def gfcc_solve_ea(h, p, omega, eta, tol, return_y=False, allow_noconv=False):
    """advanced part: G^A [nw, np, np] (host numpy); return_y: also Y1 [np*nw, v], Y2 [np*nw, o, v, v] (task r = iq*nw + iw)."""
    torch = _torch()
    pa = np.ascontiguousarray(p, dtype=np.int32)
    npn, nw = len(pa), len(np.atleast_1d(omega))
    om, omp = _omega(np.atleast_1d(omega), nw)
    G = np.empty((nw, npn, npn), dtype=np.complex128)
    allow = (GFCC_ENOCONV,) if allow_noconv else ()
    pp = pa.ctypes.data_as(ctypes.POINTER(ctypes.c_int))
    if return_y:
        Y1 = torch.empty((npn * nw, h.v), dtype=torch.complex128, device="cuda")
        Y2 = torch.empty((npn * nw, h.o, h.v, h.v), dtype=torch.complex128, device="cuda")
        _check(h, lib().gfcc_solve_ea_x(h.ptr, npn, pp, nw, omp, float(eta), float(tol), G.ctypes.data,
                                        ctypes.c_void_p(Y1.data_ptr()), ctypes.c_void_p(Y2.data_ptr())), allow)
        return G, Y1, Y2
    _check(h, lib().gfcc_solve_ea(h.ptr, npn, pp, nw, omp, float(eta), float(tol), G.ctypes.data), allow)
    return G


def gfcc_assemble_g_ea(h, Y1, Y2, p):
    torch = _torch()
    pa = np.ascontiguousarray(p, dtype=np.int32)
    nrhs = Y1.shape[0]
    G = np.empty((nrhs, len(pa)), dtype=np.complex128)
    _check(h, lib().gfcc_assemble_g_ea(h.ptr, nrhs, _dev(Y1, torch.complex128), _dev(Y2, torch.complex128), len(pa),
                                       pa.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), G.ctypes.data))
    return G


# ---- model-order reduction (Eq. 9-10; Alg. 1 lines 18-21) -----------------------------------
def gfcc_mor_reset(h, m_cap):
    _check(h, lib().gfcc_mor_reset(h.ptr, int(m_cap)))


def gfcc_mor_extend(h, X1, X2, droptol=1e-8):
    """X1 [nx,o], X2 [nx,o,o,v] complex128 CUDA tensors (e.g. from gfcc_solve_ip(..., return_x=True)) -> new dimension m."""
    torch = _torch()
    m = ctypes.c_int(0)
    _check(h, lib().gfcc_mor_extend(h.ptr, int(X1.shape[0]), _dev(X1, torch.complex128), _dev(X2, torch.complex128),
                                    float(droptol), ctypes.byref(m)))
    return m.value


def gfcc_mor_solve(h, p, omega, eta):
    """Reduced model on a frequency grid -> (G [nw,np,np] complex128, A [nw] float64), host numpy arrays."""
    _torch()
    pa = np.ascontiguousarray(p, dtype=np.int32)
    om = np.ascontiguousarray(np.atleast_1d(omega), dtype=np.float64)
    G = np.empty((len(om), len(pa), len(pa)), dtype=np.complex128)
    A = np.empty(len(om), dtype=np.float64)
    _check(h, lib().gfcc_mor_solve(h.ptr, len(pa), pa.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), len(om),
                                   om.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), float(eta), G.ctypes.data,
                                   A.ctypes.data_as(ctypes.POINTER(ctypes.c_double))))
    return G, A


def gfcc_mor_get(h, name):
    """"m"/"cap" -> int; "Hhat" -> [m,m], "S"/"HS" -> [n,m] host numpy arrays (parity hooks)."""
    n = lib().gfcc_mor_get(h.ptr, name.encode(), None)
    if n < 0:
        _check(h, int(n))
    if name in ("m", "cap"):
        return int(n)
    m = int(lib().gfcc_mor_get(h.ptr, b"m", None))
    out = np.empty(int(n), dtype=np.float64)
    if n > 0:
        n2 = lib().gfcc_mor_get(h.ptr, name.encode(), out.ctypes.data)
        if n2 < 0:
            _check(h, int(n2))
    return out.reshape(-1, m) if m > 0 else out.reshape(0, 0)
