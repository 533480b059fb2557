"""CPU oracle for the GFCCSD-IP hot path -- TEST INFRASTRUCTURE ONLY.

Thin ctypes wrapper around oracle/gfcc_oracle.cpp (plain C++ loops, FP64) plus the dense-LU
route (numpy.linalg.solve as the library step).  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg may import this package.  It never imports the
CUDA package (paper_2010_04768_b200) and shares no code with it.

Citations: PAPER.md:59-94 (Eqs. 1-8), PAPER.md:136-138 (GMRES); SURVEY.md section 8(c) for the
working equations (the paper prints none).
"""
import ctypes
import os

import numpy as np

from .build import build as _build

_c_double_p = ctypes.POINTER(ctypes.c_double)
_c_int_p = ctypes.POINTER(ctypes.c_int)


def _dp(a):
    return a.ctypes.data_as(_c_double_p)


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build()
        L = ctypes.CDLL(path)
        L.orc_create.restype = ctypes.c_void_p
        L.orc_create.argtypes = [ctypes.c_int] * 3 + [_c_double_p] * 6 + [ctypes.c_int]
        L.orc_destroy.argtypes = [ctypes.c_void_p]
        L.orc_threads.restype = ctypes.c_int
        L.orc_get.restype = ctypes.c_longlong
        L.orc_get.argtypes = [ctypes.c_void_p, ctypes.c_char_p, _c_double_p]
        L.orc_sigma.argtypes = [ctypes.c_void_p, ctypes.c_int, _c_double_p, ctypes.c_double] + [_c_double_p] * 4
        L.orc_rhs.argtypes = [ctypes.c_void_p, ctypes.c_int, _c_double_p, _c_double_p]
        L.orc_bra.argtypes = [ctypes.c_void_p, ctypes.c_int, _c_double_p, _c_double_p]
        L.orc_bra_dot.argtypes = [ctypes.c_void_p] + [_c_double_p] * 5
        L.orc_gmres.restype = ctypes.c_int
        L.orc_gmres.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                ctypes.c_int, ctypes.c_int, ctypes.c_int, _c_double_p, _c_double_p, _c_double_p]
        L.orc_gmres_hist.restype = ctypes.c_int
        L.orc_gmres_hist.argtypes = L.orc_gmres.argtypes + [_c_double_p, ctypes.c_int]
        L.orc_sigma_ea.argtypes = [ctypes.c_void_p, ctypes.c_int, _c_double_p, ctypes.c_double] + [_c_double_p] * 4
        L.orc_rhs_ea.argtypes = [ctypes.c_void_p, ctypes.c_int, _c_double_p, _c_double_p]
        L.orc_bra_ea.argtypes = [ctypes.c_void_p, ctypes.c_int, _c_double_p, _c_double_p]
        L.orc_bra_dot_ea.argtypes = [ctypes.c_void_p] + [_c_double_p] * 5
        L.orc_gmres_ea.restype = ctypes.c_int
        L.orc_gmres_ea.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                   ctypes.c_int, ctypes.c_int, ctypes.c_int, _c_double_p, _c_double_p, _c_double_p,
                                   _c_double_p, ctypes.c_int]
        L.orc_sigma_rows.argtypes = [ctypes.c_void_p, ctypes.c_int, _c_double_p, ctypes.c_double, _c_double_p,
                                     _c_double_p, ctypes.c_int, _c_int_p, _c_double_p, ctypes.c_int, _c_int_p,
                                     _c_double_p]
        _lib = L
    return _lib


def threads() -> int:
    return lib().orc_threads()


MODE_DEF = 1      # definition form (items 1-7 with explicit <pq||rs> blocks)
MODE_ROWS = 2     # T1-dressed factorised form for row-sampled sigma
MODE_EA = 4       # with MODE_DEF: EA / advanced-part intermediates (W_amef, W_abef, W_abei; O(v^4) memory)


class Oracle:
    """Inputs are host numpy float64 arrays in the C-ABI layouts (see include/gfcc.h):
    fock [N,N]; T1, L1 [o,v]; T2p [npair,v,v]; L2p [npair,ntri]; Lchol [Q,N,N]."""

    def __init__(self, o, v, Q, fock, T1, T2p, L1, L2p, Lchol, mode=MODE_DEF):
        self.o, self.v, self.Q, self.N = o, v, Q, o + v
        self.npair = o * (o - 1) // 2
        self.ntri = v * (v - 1) // 2
        c = lambda a: np.ascontiguousarray(a, dtype=np.float64)
        # keep references: the C side borrows T2p, L2p, Lchol
        self._keep = [c(fock), c(T1), c(T2p), c(L1), c(L2p), c(Lchol)]
        f, t1, t2p, l1, l2p, Lc = self._keep
        assert f.shape == (self.N, self.N) and t1.shape == (o, v) and l1.shape == (o, v)
        assert t2p.size == self.npair * v * v and l2p.size == self.npair * self.ntri and Lc.shape == (Q, self.N, self.N)
        self.mode = mode
        self.h = lib().orc_create(o, v, Q, _dp(f), _dp(t1), _dp(t2p), _dp(l1), _dp(l2p), _dp(Lc), mode)

    def __del__(self):
        if getattr(self, "h", None):
            lib().orc_destroy(self.h)
            self.h = None

    # ---- intermediates (definition form) -------------------------------------------------
    def get(self, name):
        n = lib().orc_get(self.h, name.encode(), None)
        if n < 0:
            raise KeyError(name)
        out = np.empty(n, dtype=np.float64)
        lib().orc_get(self.h, name.encode(), _dp(out))
        o, v, N = self.o, self.v, self.N
        shapes = dict(Fme=(o, v), Fmi=(o, o), Fae=(v, v), Wmnij=(o, o, o, o), Wmnie=(o, o, o, v),
                      Wmbej=(o, v, v, o), Wmbij=(o, v, o, o), oovv=(o, o, v, v), ft=(N, N),
                      Wamef=(v, o, v, v), Wabef=(v, v, v, v), Wabei=(v, v, v, o))
        return out.reshape(shapes[name])

    # ---- sigma ---------------------------------------------------------------------------
    def sigma(self, omega, eta, X1, X2):
        """Definition-form sigma. X1 [nrhs,o], X2 [nrhs,o,o,v] complex128 -> (S1, S2)."""
        X1 = np.ascontiguousarray(X1, dtype=np.complex128)
        X2 = np.ascontiguousarray(X2, dtype=np.complex128)
        nrhs = X1.shape[0]
        om = np.ascontiguousarray(np.broadcast_to(np.asarray(omega, dtype=np.float64), (nrhs,)))
        S1 = np.empty_like(X1)
        S2 = np.empty_like(X2)
        rc = lib().orc_sigma(self.h, nrhs, _dp(om), float(eta), _dp(X1.view(np.float64)), _dp(X2.view(np.float64)),
                             _dp(S1.view(np.float64)), _dp(S2.view(np.float64)))
        if rc:
            raise RuntimeError("orc_sigma needs MODE_DEF")
        return S1, S2

    def sigma_rows(self, omega, eta, X1, X2, s1_idx, s2_idx):
        """Row-sampled sigma: returns (S1[len(s1_idx), nrhs], S2[len(s2_idx), nrhs])."""
        X1 = np.ascontiguousarray(X1, dtype=np.complex128)
        X2 = np.ascontiguousarray(X2, dtype=np.complex128)
        nrhs = X1.shape[0]
        om = np.ascontiguousarray(np.broadcast_to(np.asarray(omega, dtype=np.float64), (nrhs,)))
        i1 = np.ascontiguousarray(s1_idx, dtype=np.int32).reshape(-1)
        i2 = np.ascontiguousarray(s2_idx, dtype=np.int32).reshape(-1, 3)
        S1 = np.empty((len(i1), nrhs), dtype=np.complex128)
        S2 = np.empty((len(i2), nrhs), dtype=np.complex128)
        rc = lib().orc_sigma_rows(self.h, nrhs, _dp(om), float(eta), _dp(X1.view(np.float64)),
                                  _dp(X2.view(np.float64)), len(i1), i1.ctypes.data_as(_c_int_p),
                                  _dp(S1.view(np.float64)), len(i2), i2.ctypes.data_as(_c_int_p),
                                  _dp(S2.view(np.float64)))
        if rc:
            raise RuntimeError("orc_sigma_rows needs MODE_ROWS")
        return S1, S2

    # ---- b_p, c_q ------------------------------------------------------------------------
    def rhs(self, p):
        b1 = np.empty(self.o, dtype=np.complex128)
        b2 = np.empty((self.o, self.o, self.v), dtype=np.complex128)
        if lib().orc_rhs(self.h, int(p), _dp(b1.view(np.float64)), _dp(b2.view(np.float64))):
            raise ValueError("p out of range")
        return b1, b2

    def bra(self, q):
        c1 = np.empty(self.o)
        c2 = np.empty((self.o, self.o, self.v))
        if lib().orc_bra(self.h, int(q), _dp(c1), _dp(c2)):
            raise ValueError("q out of range")
        return c1, c2

    def bra_dot(self, c1, c2, x1, x2):
        out = np.empty(1, dtype=np.complex128)
        x1 = np.ascontiguousarray(x1, dtype=np.complex128)
        x2 = np.ascontiguousarray(x2, dtype=np.complex128)
        lib().orc_bra_dot(self.h, _dp(c1), _dp(c2), _dp(x1.view(np.float64)), _dp(x2.view(np.float64)),
                          _dp(out.view(np.float64)))
        return out[0]

    # ---- packing helpers (packed 1h + 2h1p(i<j) basis) -------------------------------------
    def pack(self, x1, x2):
        iu = np.triu_indices(self.o, 1)
        return np.concatenate([np.asarray(x1).reshape(-1), np.asarray(x2)[iu[0], iu[1], :].reshape(-1)])

    def unpack(self, z):
        o, v = self.o, self.v
        x1 = z[:o].copy()
        x2 = np.zeros((o, o, v), dtype=z.dtype)
        iu = np.triu_indices(o, 1)
        blk = z[o:].reshape(-1, v)
        x2[iu[0], iu[1], :] = blk
        x2[iu[1], iu[0], :] = -blk
        return x1, x2

    # ---- solves --------------------------------------------------------------------------
    def gmres(self, p, omega, eta, tol, m=50, maxit=1000, x0kind=1, history=False):
        """GMRES(m) for one (p, omega). Returns (x1, x2, n_sigma_applications, relres[, hist]); hist[k] = relative residual
        (estimate) after sigma application k+1."""
        x1 = np.empty(self.o, dtype=np.complex128)
        x2 = np.empty((self.o, self.o, self.v), dtype=np.complex128)
        rr = np.empty(1)
        hist = np.full(int(maxit) + 1, np.nan)
        n = lib().orc_gmres_hist(self.h, int(p), float(omega), float(eta), float(tol), int(m), int(maxit), int(x0kind),
                                 _dp(x1.view(np.float64)), _dp(x2.view(np.float64)), _dp(rr), _dp(hist), len(hist))
        if n < 0:
            raise RuntimeError("orc_gmres needs MODE_DEF")
        if history:
            return x1, x2, n, rr[0], hist[:n]
        return x1, x2, n, rr[0]

    def dense_hbar(self):
        """Real matrix of Hbar_IP in the packed basis: column nu = sigma(e_nu) at omega = eta = 0."""
        n = self.o + self.npair * self.v
        H = np.empty((n, n))
        bs = 64
        for c0 in range(0, n, bs):
            c1 = min(n, c0 + bs)
            X1 = np.zeros((c1 - c0, self.o), dtype=np.complex128)
            X2 = np.zeros((c1 - c0, self.o, self.o, self.v), dtype=np.complex128)
            for k in range(c0, c1):
                e = np.zeros(n, dtype=np.complex128)
                e[k] = 1.0
                X1[k - c0], X2[k - c0] = self.unpack(e)
            S1, S2 = self.sigma(0.0, 0.0, X1, X2)
            for k in range(c0, c1):
                H[:, k] = self.pack(S1[k - c0], S2[k - c0]).real
        return H

    def G_dense(self, plist, omegas, eta, H=None):
        """G[w, ip, iq] = c_q^T ((omega - i eta) 1 + Hbar_IP)^-1 b_p by dense LU (numpy.linalg.solve)."""
        if H is None:
            H = self.dense_hbar()
        n = H.shape[0]
        B = np.stack([self.pack(*self.rhs(p)) for p in plist], axis=1)
        C = np.stack([self.pack(*self.bra(q)) for q in plist], axis=1)
        G = np.empty((len(omegas), len(plist), len(plist)), dtype=np.complex128)
        for iw, w in enumerate(omegas):
            X = np.linalg.solve(H + (w - 1j * eta) * np.eye(n), B)
            G[iw] = (C.T @ X).T          # [ip, iq]
        return G

    # ---- EA / advanced part (Eq. 6; second terms of Eq. 7-8) ---------------------------------
    # vectors: y1 [v], y2 [o, v, v] (index order j, a, b; antisymmetric in a, b); packed basis: 1p then (j, a<b), j slowest
    def sigma_ea(self, omega, eta, Y1, Y2):
        """sigma_EA = (omega + i eta) Y - Hbar Y.  Y1 [nrhs,v], Y2 [nrhs,o,v,v] complex128 -> (S1, S2)."""
        Y1 = np.ascontiguousarray(Y1, dtype=np.complex128)
        Y2 = np.ascontiguousarray(Y2, dtype=np.complex128)
        nrhs = Y1.shape[0]
        om = np.ascontiguousarray(np.broadcast_to(np.asarray(omega, dtype=np.float64), (nrhs,)))
        S1 = np.empty_like(Y1)
        S2 = np.empty_like(Y2)
        rc = lib().orc_sigma_ea(self.h, nrhs, _dp(om), float(eta), _dp(Y1.view(np.float64)), _dp(Y2.view(np.float64)),
                                _dp(S1.view(np.float64)), _dp(S2.view(np.float64)))
        if rc:
            raise RuntimeError("orc_sigma_ea needs MODE_DEF | MODE_EA")
        return S1, S2

    def rhs_ea(self, q):
        b1 = np.empty(self.v, dtype=np.complex128)
        b2 = np.empty((self.o, self.v, self.v), dtype=np.complex128)
        if lib().orc_rhs_ea(self.h, int(q), _dp(b1.view(np.float64)), _dp(b2.view(np.float64))):
            raise ValueError("q out of range")
        return b1, b2

    def bra_ea(self, p):
        c1 = np.empty(self.v)
        c2 = np.empty((self.o, self.v, self.v))
        if lib().orc_bra_ea(self.h, int(p), _dp(c1), _dp(c2)):
            raise ValueError("p out of range")
        return c1, c2

    def bra_dot_ea(self, c1, c2, y1, y2):
        out = np.empty(1, dtype=np.complex128)
        y1 = np.ascontiguousarray(y1, dtype=np.complex128)
        y2 = np.ascontiguousarray(y2, dtype=np.complex128)
        lib().orc_bra_dot_ea(self.h, _dp(c1), _dp(c2), _dp(y1.view(np.float64)), _dp(y2.view(np.float64)),
                             _dp(out.view(np.float64)))
        return out[0]

    def pack_ea(self, y1, y2):
        au = np.triu_indices(self.v, 1)
        return np.concatenate([np.asarray(y1).reshape(-1), np.asarray(y2)[:, au[0], au[1]].reshape(-1)])

    def unpack_ea(self, z):
        o, v = self.o, self.v
        y1 = z[:v].copy()
        y2 = np.zeros((o, v, v), dtype=z.dtype)
        au = np.triu_indices(v, 1)
        blk = z[v:].reshape(o, -1)
        y2[:, au[0], au[1]] = blk
        y2[:, au[1], au[0]] = -blk
        return y1, y2

    def gmres_ea(self, q, omega, eta, tol, m=50, maxit=1000, x0kind=1, history=False):
        y1 = np.empty(self.v, dtype=np.complex128)
        y2 = np.empty((self.o, self.v, self.v), dtype=np.complex128)
        rr = np.empty(1)
        hist = np.full(int(maxit) + 1, np.nan)
        n = lib().orc_gmres_ea(self.h, int(q), float(omega), float(eta), float(tol), int(m), int(maxit), int(x0kind),
                               _dp(y1.view(np.float64)), _dp(y2.view(np.float64)), _dp(rr), _dp(hist), len(hist))
        if n < 0:
            raise RuntimeError("orc_gmres_ea needs MODE_DEF | MODE_EA")
        return (y1, y2, n, rr[0], hist[:n]) if history else (y1, y2, n, rr[0])

    def dense_hbar_ea(self):
        """Real matrix of Hbar_EA in the packed basis: column nu = -(sigma_EA(e_nu) at omega = eta = 0)."""
        n = self.v + self.o * self.ntri
        H = np.empty((n, n))
        bs = 64
        for c0 in range(0, n, bs):
            c1 = min(n, c0 + bs)
            Y1 = np.zeros((c1 - c0, self.v), dtype=np.complex128)
            Y2 = np.zeros((c1 - c0, self.o, self.v, self.v), dtype=np.complex128)
            for k in range(c0, c1):
                e = np.zeros(n, dtype=np.complex128)
                e[k] = 1.0
                Y1[k - c0], Y2[k - c0] = self.unpack_ea(e)
            S1, S2 = self.sigma_ea(0.0, 0.0, Y1, Y2)
            for k in range(c0, c1):
                H[:, k] = -self.pack_ea(S1[k - c0], S2[k - c0]).real
        return H

    def G_dense_ea(self, plist, omegas, eta, H=None):
        """advanced part G^A[w, ip, iq] = c_p^T ((omega + i eta) 1 - Hbar_EA)^-1 b_q by dense LU (second term of Eq. 2 / 8)."""
        if H is None:
            H = self.dense_hbar_ea()
        n = H.shape[0]
        B = np.stack([self.pack_ea(*self.rhs_ea(q)) for q in plist], axis=1)
        C = np.stack([self.pack_ea(*self.bra_ea(p)) for p in plist], axis=1)
        G = np.empty((len(omegas), len(plist), len(plist)), dtype=np.complex128)
        for iw, w in enumerate(omegas):
            Y = np.linalg.solve((w + 1j * eta) * np.eye(n) - H, B)      # columns q
            G[iw] = C.T @ Y                                              # [ip, iq]
        return G
