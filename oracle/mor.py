"""CPU oracle for the model-order-reduction (MOR) step of the GFCC workflow -- TEST INFRASTRUCTURE ONLY.

Follows the paper step by step (Eq. 10; Alg. 1 lines 18-21 `PAPER.md:225-228`):
  (i)  Gram-Schmidt of the newly obtained X_p(omega) against the previous orthonormal vectors -> S = {v_1..v_m};
  (ii) projection  H^ = S^T Hbar_N S,  b^ = S^T b,  c^T^ = c^T S;
  (iii) solve (omega - i eta + H^) X^ = b^ for every omega of the fine grid,  G^ = c^^T X^,
        A(omega) = (1/pi) sum_p Im G^_pp  (Eq. 9; sign: see below).
Reading (item 24): Eq. 10 writes TRANSPOSES throughout and Hbar, b, c are real, so S is a real
orthonormal basis: every complex X contributes its real and its imaginary part, in the order Re X_0, Im X_0, Re X_1, ...
Sign of Eq. 9 (reading 25): the paper prints A = -(1/pi) Tr Im G^R, which is non-negative for a +i eta regularisation;
its own Eq. 2/5 use (omega + Hbar_N - i eta) for the IP part, for which Im G_pp = +eta/((omega-eps_p)^2+eta^2) >= 0 at
zeroth order.  A spectral function is non-negative, so with Eq. 5's sign A = +(1/pi) sum_p Im G_pp.
Each candidate is normalised, orthogonalised twice (classical Gram-Schmidt with re-orthogonalisation) against all vectors
accepted so far and dropped when what is left of its unit norm is <= droptol.  Plain numpy in FP64; numpy.linalg.solve is
the library step.  Shares no code with the CUDA path.
"""
import numpy as np


def mor_extend(S, X, droptol=1e-8):
    """S: (n, m) real orthonormal columns or None; X: (k, n) complex packed vectors (1h + 2h1p(i<j) basis, the metric of
    DESIGN.md reading 9).  Returns the extended basis (n, m')."""
    X = np.atleast_2d(np.asarray(X, dtype=np.complex128))
    n = X.shape[1]
    cols = [] if S is None else [S[:, j].copy() for j in range(S.shape[1])]
    for r in range(X.shape[0]):
        for part in (X[r].real, X[r].imag):
            v = np.array(part, dtype=np.float64)
            nrm = np.sqrt(np.dot(v, v))
            if nrm == 0.0:
                continue
            v /= nrm
            for _ in range(2):
                if cols:
                    B = np.stack(cols, axis=1)
                    v = v - B @ (B.T @ v)
            nrm = np.sqrt(np.dot(v, v))
            if nrm > droptol:
                cols.append(v / nrm)
    if not cols:
        return np.zeros((n, 0))
    return np.stack(cols, axis=1)


def mor_project(H, S, B, C):
    """H (n,n) real Hbar_IP; B (n,np) right-hand sides b_p; C (n,nq) bra vectors c_q -> (H^, b^, c^)  (Eq. 10)."""
    return S.T @ (H @ S), S.T @ B, S.T @ C


def mor_green(Hh, bh, ch, omegas, eta):
    """G^[w, ip, iq] = c^_q^T (omega - i eta + H^)^-1 b^_p and A[w] = (1/pi) sum_p Im G^[w,p,p]  (Eq. 9-10)."""
    m = Hh.shape[0]
    omegas = np.atleast_1d(omegas)
    G = np.empty((len(omegas), bh.shape[1], ch.shape[1]), dtype=np.complex128)
    for iw, w in enumerate(omegas):
        Xh = np.linalg.solve(Hh + (w - 1j * eta) * np.eye(m), bh.astype(np.complex128))
        G[iw] = (ch.T @ Xh).T
    A = np.einsum("wpp->w", G.imag) / np.pi
    return G, A
