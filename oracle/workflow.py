"""CPU oracle for the level loop of the retarded GFCCSD workflow (Alg. 1) -- TEST INFRASTRUCTURE ONLY.

Follows Alg. 1 line by line with exact (dense LU) solves in place of GMRES:
  levels -> frequencies of the level -> X_p(omega) for every target p (Eq. 5) -> Gram-Schmidt of the level's
  solutions into the subspace S (line 18) -> projection (line 19) -> spectral function on the fine grid (line 20, Eq. 9-10)
  -> "determine convergence (OR) list of frequencies to be processed in next level" (line 21).
Frequencies are sampled by "the adaptive midpoint refinement strategy described in Ref. 100", which the
paper does not restate; Eq. 12-13 fix its counts.  Reading (items 26-27):
  * fine grid  w_k = w_min + k dw,  k = 0 .. N_tot-1,  N_tot = (w_max - w_min)/dw + 1;
  * level 1 samples 3 points (Eq. 12): both ends and the middle grid point;
  * level L > 1 samples the middle grid points of intervals between neighbouring sampled points, at most 2^(L-1) of them
    (Eq. 12).  Level 2 takes every interval (there is no earlier model to compare with); later levels take the intervals on
    which the fine-grid spectral function moved by more than spec_tol * max(A) between the two latest models, largest
    change first;
  * converged when no interval qualifies (or none can be split); never more than L_max = floor(log2((w_max-w_min)/dw))
    levels (Eq. 13).
Plain numpy; uses oracle/mor.py for the MOR steps.  Shares no code with the CUDA path.
"""
import math

import numpy as np

from . import mor


def fine_grid(wmin, wmax, dw):
    n_tot = int(round((wmax - wmin) / dw)) + 1
    return wmin + dw * np.arange(n_tot)


def level_bound(wmin, wmax, dw):
    """Eq. 13: L_max <= log2((w_max - w_min) / dw)"""
    return max(1, int(math.floor(math.log2((wmax - wmin) / dw) + 1e-12)))


def next_level_points(sampled, A_new, A_old, level_next, spec_tol):
    """grid indices to sample at level `level_next` (>= 2).  sampled: sorted grid indices already used."""
    cap = 2 ** (level_next - 1)                                   # Eq. 12
    scale = max(float(np.abs(A_new).max()), 1e-300)
    cand = []
    for a, b in zip(sampled[:-1], sampled[1:]):
        if b - a < 2:
            continue
        if A_old is None:
            d = np.inf
        else:
            d = float(np.abs(A_new[a:b + 1] - A_old[a:b + 1]).max()) / scale
            if d <= spec_tol:
                continue
        cand.append((d, a, b))
    cand.sort(key=lambda t: (-t[0], t[1]))                        # largest change first, then left to right
    return sorted((a + b) // 2 for _, a, b in cand[:cap])


def run(H, B, C, wmin, wmax, dw, eta, spec_tol=1e-3, max_levels=0, droptol=1e-8):
    """H (n,n) real Hbar_IP, B (n,np) right-hand sides b_p, C (n,np) bra vectors c_q.
    Returns dict(w, A, G, level_of, levels, m): fine grid, final spectral function and reduced G^ on it, the level at which
    each grid point was sampled (0 = never), number of levels run, final subspace dimension."""
    w = fine_grid(wmin, wmax, dw)
    n_tot = len(w)
    n = H.shape[0]
    lmax = level_bound(wmin, wmax, dw)
    if max_levels > 0:
        lmax = min(lmax, max_levels)
    level_of = np.zeros(n_tot, dtype=np.int32)
    new = sorted({0, (n_tot - 1) // 2, n_tot - 1})
    S, A_old, A_new, G_new = None, None, None, None
    level = 0
    eye = np.eye(n)
    while new:
        level += 1
        for k in new:
            level_of[k] = level
        # Alg. 1 lines 4-16: X_p(omega) for every target p, here by LU (order p-major like the C ABI: r = ip*nw + iw)
        sols = [np.linalg.solve(H + (w[k] - 1j * eta) * eye, B.astype(np.complex128)) for k in new]      # each (n, np)
        X = np.stack([sols[iw][:, ip] for ip in range(B.shape[1]) for iw in range(len(new))], axis=0)
        S = mor.mor_extend(S, X, droptol)                                                                 # line 18
        Hh, bh, ch = mor.mor_project(H, S, B, C)                                                          # line 19
        G_new, A_new = mor.mor_green(Hh, bh, ch, w, eta)                                                  # line 20
        if level >= lmax:
            break
        sampled = sorted(int(k) for k in np.nonzero(level_of)[0])
        new = next_level_points(sampled, A_new, A_old, level + 1, spec_tol)                               # line 21
        A_old = A_new
    return {"w": w, "A": A_new, "G": G_new, "level_of": level_of, "levels": level, "m": S.shape[1]}
