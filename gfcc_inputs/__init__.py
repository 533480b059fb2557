"""Seeded synthetic inputs for the GFCCSD-IP hot path (shared by the oracle tests and the CUDA path).

This module holds NONE of the method's arithmetic: it only draws numbers.  Every tensor element is a
pure function of (seed, tensor id, canonical element index) through a counter-based 32-bit integer
hash, so any slice can be regenerated independently; values are produced with torch element-wise
ops and can be generated on the CPU or directly in device memory (large configs).  CPU- and
GPU-generated normals may differ in the last ulp (log/cos), therefore a test always materialises a
tensor ONCE and hands the same bits to both sides.

The five configs are BASELINE.json:configs[0..4]; they stand in for the paper's molecular workloads
(C60/cc-pVDZ shape at config 4), whose integrals and amplitudes are not available.
Readings of the config text (SURVEY.md 8c points 12-16) are restated in DESIGN.md "Input recipe".
"""
import math

import torch

SEED0 = 20201004

#            o    v    Q     np  nw  w_lo  w_hi   tol    nrhs (np*nw)
CONFIGS = {
    0: dict(o=8, v=24, Q=96, np=4, nw=8, wlo=-1.0, whi=-0.2, eta=0.01, tol=1e-10),
    1: dict(o=40, v=160, Q=600, np=16, nw=16, wlo=-1.2, whi=-0.2, eta=0.01, tol=1e-8),
    2: dict(o=80, v=320, Q=1200, np=16, nw=4, wlo=-1.0, whi=-0.25, eta=0.01, tol=1e-8),
    3: dict(o=120, v=480, Q=1800, np=8, nw=4, wlo=-1.0, whi=-0.25, eta=0.01, tol=1e-8),
    4: dict(o=180, v=660, Q=2500, np=4, nw=4, wlo=-1.0, whi=-0.25, eta=0.01, tol=1e-8),
}

# tensor ids
TID_EPS_O, TID_EPS_V, TID_L, TID_T1, TID_L1, TID_T2, TID_L2, TID_X1, TID_X2, TID_Y1, TID_Y2 = range(1, 12)

_M32 = 0xFFFFFFFF


def _mul32(x, c):
    """(x * c) mod 2^32 for int64 tensors holding values < 2^32, without 64-bit overflow."""
    lo = (x & 0xFFFF) * c
    hi = (((x >> 16) * c) & 0xFFFF) << 16
    return (lo + hi) & _M32


def _mix32(x):
    x = x ^ (x >> 16)
    x = _mul32(x, 0x7FEB352D)
    x = x ^ (x >> 15)
    x = _mul32(x, 0x846CA68B)
    x = x ^ (x >> 16)
    return x


def _hash(seed, tid, idx):
    """idx: int64 tensor of non-negative canonical indices (< 2^62) -> int64 tensor of 32-bit hashes."""
    key = (int(seed) * 0x9E3779B1 + int(tid) * 0x85EBCA77) & _M32
    lo = idx & _M32
    hi = (idx >> 32) & _M32
    h = _mix32(hi ^ key)
    h = _mix32(lo ^ h)
    return h


def uniform(seed, tid, idx):
    """float64 in (0,1), 53-bit, from two decorrelated 32-bit hashes."""
    h = _hash(seed, tid, idx)
    h1 = _mix32(h ^ 0x68E31DA4)
    h2 = _mix32(h ^ 0xB5297A4D)
    m = (h1 >> 5) * 67108864 + (h2 >> 6)          # 27 + 26 bits
    return (m.to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal(seed, tid, idx):
    """standard normal via Box-Muller on two uniforms keyed by the same canonical index."""
    u1 = uniform(seed, tid, idx * 2)
    u2 = uniform(seed, tid, idx * 2 + 1)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)


def _arange(n, device, start=0):
    return torch.arange(start, start + n, dtype=torch.int64, device=device)


def npair(o):
    return o * (o - 1) // 2


def ntri(v):
    return v * (v - 1) // 2


def pair_index(i, j, o):
    """index of the pair (i<j) in the packed order used everywhere: i*o - i(i+1)/2 + (j-i-1)."""
    return i * o - i * (i + 1) // 2 + (j - i - 1)


def seed_of(cfg_id):
    return SEED0 + int(cfg_id)


# ------------------------------------------------------------------------------------------
def orbital_energies(o, v, seed, banded=False, device="cpu"):
    """occ eps ~ U[-1.5,-0.3], virt eps ~ U[0.1,3.0] (sorted).  banded (config 4): occupied levels in
    [-1.0,-0.25] as o/5 equally spaced group centres, 5 members split by (-2,-1,0,1,2)*1e-3 Ha."""
    if banded:
        ng = (o + 4) // 5
        centres = torch.linspace(-1.0, -0.25, ng, dtype=torch.float64, device=device)
        split = torch.tensor([-2.0, -1.0, 0.0, 1.0, 2.0], dtype=torch.float64, device=device) * 1e-3
        eo = (centres[:, None] + split[None, :]).reshape(-1)[:o]
    else:
        eo = -1.5 + 1.2 * uniform(seed, TID_EPS_O, _arange(o, device))
    ev = 0.1 + 2.9 * uniform(seed, TID_EPS_V, _arange(v, device))
    return torch.sort(eo)[0], torch.sort(ev)[0]


def fock(o, v, seed, banded=False, device="cpu"):
    eo, ev = orbital_energies(o, v, seed, banded, device)
    return torch.diag(torch.cat([eo, ev]))


def cholesky(o, v, Q, seed, device="cpu", scale=1.0):
    """L[q,p,r] = g * exp(-q/30) / sqrt(Q), g ~ N(0,1) keyed by (q, min(p,r), max(p,r)): symmetric in (p,r)."""
    N = o + v
    out = torch.empty((Q, N, N), dtype=torch.float64, device=device)
    p = _arange(N, device)
    lo = torch.minimum(p[:, None], p[None, :])
    hi = torch.maximum(p[:, None], p[None, :])
    canon = lo * N + hi
    for q in range(Q):
        g = normal(seed, TID_L, canon + q * N * N)
        out[q] = g * (scale * math.exp(-q / 30.0) / math.sqrt(Q))
    return out


def singles(o, v, seed, tid, sigma=0.01, device="cpu"):
    return sigma * normal(seed, tid, _arange(o * v, device)).reshape(o, v)


def doubles_pairpacked(o, v, seed, tid, sigma=0.02, device="cpu", out=None, chunk_pairs=None):
    """[npair][v][v], antisymmetric in (a,b): canonical element (pair, a<b) ~ N(0, sigma)."""
    P = npair(o)
    if out is None:
        out = torch.empty((P, v, v), dtype=torch.float64, device=device)
    if chunk_pairs is None:
        chunk_pairs = max(1, (1 << 24) // (v * v))
    a = _arange(v, device)
    lo = torch.minimum(a[:, None], a[None, :])
    hi = torch.maximum(a[:, None], a[None, :])
    canon = (lo * v + hi)[None, :, :]
    sign = torch.sign((a[None, :] - a[:, None]).to(torch.float64))[None, :, :]     # +1 for a<b, -1 for a>b, 0 diag
    for p0 in range(0, P, chunk_pairs):
        p1 = min(P, p0 + chunk_pairs)
        pid = _arange(p1 - p0, device, p0)[:, None, None]
        g = normal(seed, tid, pid * (v * v) + canon)
        out[p0:p1] = sigma * g * sign
    return out


def doubles_fullpacked(o, v, seed, tid, sigma=0.02, device="cpu", out=None, chunk_pairs=None):
    """[npair][ntri]: the a<b triangle of the same tensor doubles_pairpacked(...) would give."""
    P, T = npair(o), ntri(v)
    if out is None:
        out = torch.empty((P, T), dtype=torch.float64, device=device)
    if chunk_pairs is None:
        chunk_pairs = max(1, (1 << 24) // max(T, 1))
    iu = torch.triu_indices(v, v, 1, device=device)
    canon = (iu[0] * v + iu[1])[None, :]
    for p0 in range(0, P, chunk_pairs):
        p1 = min(P, p0 + chunk_pairs)
        pid = _arange(p1 - p0, device, p0)[:, None]
        out[p0:p1] = sigma * normal(seed, tid, pid * (v * v) + canon)
    return out


def trial_vectors(o, v, nrhs, seed, device="cpu"):
    """X1 [nrhs,o], X2 [nrhs,o,o,v] complex128 ~ N(0,1)+iN(0,1), X2 antisymmetrised in (i,j)."""
    x1 = normal(seed, TID_X1, _arange(nrhs * o * 2, device)).reshape(nrhs, o, 2)
    X1 = torch.complex(x1[..., 0], x1[..., 1])
    X2 = torch.zeros((nrhs, o, o, v), dtype=torch.complex128, device=device)
    iu = torch.triu_indices(o, o, 1, device=device)
    P = iu.shape[1]
    for r in range(nrhs):
        g = normal(seed, TID_X2, _arange(P * v * 2, device, r * P * v * 2)).reshape(P, v, 2)
        z = torch.complex(g[..., 0], g[..., 1])
        X2[r, iu[0], iu[1], :] = z
        X2[r, iu[1], iu[0], :] = -z
    return X1, X2


def trial_vectors_ea(o, v, nrhs, seed, device="cpu"):
    """EA-type trial vectors (Eq. 4): Y1 [nrhs,v], Y2 [nrhs,o,v,v] complex128 ~ N(0,1)+iN(0,1), Y2 antisymmetrised in
    (a,b); canonical element (r, j, a<b)."""
    y1 = normal(seed, TID_Y1, _arange(nrhs * v * 2, device)).reshape(nrhs, v, 2)
    Y1 = torch.complex(y1[..., 0], y1[..., 1])
    Y2 = torch.zeros((nrhs, o, v, v), dtype=torch.complex128, device=device)
    au = torch.triu_indices(v, v, 1, device=device)
    T = au.shape[1]
    for r in range(nrhs):
        g = normal(seed, TID_Y2, _arange(o * T * 2, device, r * o * T * 2)).reshape(o, T, 2)
        z = torch.complex(g[..., 0], g[..., 1])
        Y2[r][:, au[0], au[1]] = z
        Y2[r][:, au[1], au[0]] = -z
    return Y1, Y2


def omega_grid(cfg):
    c = CONFIGS[cfg] if not isinstance(cfg, dict) else cfg
    return torch.linspace(c["wlo"], c["whi"], c["nw"], dtype=torch.float64)


def targets(cfg):
    """the np highest occupied orbitals o-1, o-2, ... (near-valence focus)."""
    c = CONFIGS[cfg] if not isinstance(cfg, dict) else cfg
    return [c["o"] - 1 - k for k in range(c["np"])]


def make_system(o, v, Q, seed, device="cpu", banded=False, t1_sigma=0.01, t2_sigma=0.02, l_scale=1.0):
    """All method inputs in the C-ABI layouts: dict(fock, T1, T2p, L1, L2p, Lchol)."""
    return dict(
        o=o, v=v, Q=Q,
        fock=fock(o, v, seed, banded, device),
        T1=singles(o, v, seed, TID_T1, t1_sigma, device),
        L1=singles(o, v, seed, TID_L1, t1_sigma, device),
        T2p=doubles_pairpacked(o, v, seed, TID_T2, t2_sigma, device),
        L2p=doubles_fullpacked(o, v, seed, TID_L2, t2_sigma, device),
        Lchol=cholesky(o, v, Q, seed, device, l_scale),
    )


def make_config(cfg_id, device="cpu"):
    c = CONFIGS[cfg_id]
    s = make_system(c["o"], c["v"], c["Q"], seed_of(cfg_id), device, banded=(cfg_id == 4))
    s.update(cfg=cfg_id, eta=c["eta"], tol=c["tol"], omegas=omega_grid(cfg_id), targets=targets(cfg_id))
    return s
