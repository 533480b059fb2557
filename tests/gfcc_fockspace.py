"""Fock-space brute force for tiny systems (test-side pin of the oracle; SURVEY.md 8c pin (e)).

Independent of oracle/ and of the CUDA path: builds second-quantised operators as explicit
Jordan-Wigner matrices on 2^(o+v) determinants and evaluates the paper's operator definitions
literally (Eqs. 1-8):
    H      = sum h_pq a+_p a_q + 1/4 sum <pq||rs> a+_p a+_q a_s a_r,  h = f - sum_k <pk||qk>
    T      = sum t[i,a] a+_a a_i + 1/4 sum t[i,j,a,b] a+_a a+_b a_j a_i
    Lambda = sum l[i,a] a+_i a_a + 1/4 sum l[i,j,a,b] a+_i a+_j a_b a_a
    Hbar   = exp(-T) H_N exp(T)
    basis  tau_i = a_i, tau_ija = a+_a a_j a_i (i<j)            (Eq. 3 operator order)
    Hbar_IP[mu,nu] = <Phi| tau_mu^+ [Hbar, tau_nu] |Phi>        (connected action, reading 5)
    b_p[mu] = <Phi| tau_mu^+ exp(-T) a_p exp(T) |Phi>           (Eq. 5 rhs)
    c_q[nu] = <Phi| (1+Lambda) exp(-T) a+_q exp(T) tau_nu |Phi>  (Eq. 7 first term)
"""
import numpy as np
from scipy.linalg import expm


def jw_annihilators(n):
    Z = np.diag([1.0, -1.0])
    A = np.array([[0.0, 1.0], [0.0, 0.0]])
    I = np.eye(2)
    ops = []
    for p in range(n):
        m = np.array([[1.0]])
        for q in range(n):
            m = np.kron(m, Z if q < p else (A if q == p else I))
        ops.append(m)
    return ops


def antisym_integrals(L):
    g = np.einsum("Qpr,Qqs->pqrs", L, L)
    return g - g.transpose(0, 1, 3, 2)


def operators(o, v, f, L, t1, t2, l1, l2):
    """Jordan-Wigner matrices of everything the projections below need: (a, ad, phi, Hbar, Lam, emT, eT)."""
    N = o + v
    a = jw_annihilators(N)
    ad = [x.T for x in a]
    dim = 2 ** N
    W = antisym_integrals(L)
    h = f - np.einsum("pkqk->pq", W[:, :o, :, :o])
    H = np.zeros((dim, dim))
    for p in range(N):
        for q in range(N):
            H += h[p, q] * ad[p] @ a[q]
    for p in range(N):
        for q in range(N):
            apq = ad[p] @ ad[q]
            for r in range(N):
                for s in range(N):
                    if W[p, q, r, s] != 0.0:
                        H += 0.25 * W[p, q, r, s] * apq @ a[s] @ a[r]
    vac = np.zeros(dim)
    vac[0] = 1.0
    phi = vac.copy()
    for p in reversed(range(o)):
        phi = ad[p] @ phi
    HN = H - (phi @ H @ phi) * np.eye(dim)
    T = np.zeros((dim, dim))
    Lam = np.zeros((dim, dim))
    for i in range(o):
        for aa in range(v):
            T += t1[i, aa] * ad[o + aa] @ a[i]
            Lam += l1[i, aa] * ad[i] @ a[o + aa]
    for i in range(o):
        for j in range(o):
            for aa in range(v):
                for bb in range(v):
                    T += 0.25 * t2[i, j, aa, bb] * ad[o + aa] @ ad[o + bb] @ a[j] @ a[i]
                    Lam += 0.25 * l2[i, j, aa, bb] * ad[i] @ ad[j] @ a[o + bb] @ a[o + aa]
    eT, emT = expm(T), expm(-T)
    Hbar = emT @ HN @ eT
    return a, ad, phi, Hbar, Lam, emT, eT


def brute_force(o, v, f, L, t1, t2, l1, l2, ops=None):
    """returns H_IP [n,n], b [N,n], c [N,n] in the packed basis (1h then (i<j,a) row-major)."""
    N = o + v
    a, ad, phi, Hbar, Lam, emT, eT = ops if ops is not None else operators(o, v, f, L, t1, t2, l1, l2)
    dim = 2 ** N
    taus = [a[i] for i in range(o)]
    for i in range(o):
        for j in range(i + 1, o):
            for aa in range(v):
                taus.append(ad[o + aa] @ a[j] @ a[i])
    n = len(taus)
    HIP = np.zeros((n, n))
    for mu in range(n):
        bra = phi @ taus[mu].T
        for nu in range(n):
            HIP[mu, nu] = bra @ (Hbar @ taus[nu] - taus[nu] @ Hbar) @ phi
    bs = np.zeros((N, n))
    cs = np.zeros((N, n))
    onepl = np.eye(dim) + Lam
    for p in range(N):
        abar = emT @ a[p] @ eT
        adbar = emT @ ad[p] @ eT
        for mu in range(n):
            bs[p, mu] = phi @ taus[mu].T @ abar @ phi
            cs[p, mu] = phi @ onepl @ adbar @ taus[mu] @ phi
    return HIP, bs, cs


def brute_force_ea(o, v, f, L, t1, t2, l1, l2, ops=None):
    """Advanced (electron-attached) part, Eq. 4, Eq. 6, second terms of Eq. 7-8:
        basis  tau_a = a+_a, tau_jab = a+_a a+_b a_j (a<b)          (Eq. 4 operator order)
        Hbar_EA[mu,nu] = <Phi| tau_mu^+ [Hbar, tau_nu] |Phi>        (connected action, reading 5)
        b_q[mu] = <Phi| tau_mu^+ exp(-T) a+_q exp(T) |Phi>          (Eq. 6 rhs)
        c_p[nu] = <Phi| (1+Lambda) exp(-T) a_p exp(T) tau_nu |Phi>   (Eq. 7 second term)
    returns H_EA [n,n], b [N,n], c [N,n] in the packed basis (1p, then (j, a<b) row-major: j slowest)."""
    N = o + v
    a, ad, phi, Hbar, Lam, emT, eT = ops if ops is not None else operators(o, v, f, L, t1, t2, l1, l2)
    dim = 2 ** N
    taus = [ad[o + aa] for aa in range(v)]
    for j in range(o):
        for aa in range(v):
            for bb in range(aa + 1, v):
                taus.append(ad[o + aa] @ ad[o + bb] @ a[j])
    n = len(taus)
    HEA = np.zeros((n, n))
    for mu in range(n):
        bra = phi @ taus[mu].T
        for nu in range(n):
            HEA[mu, nu] = bra @ (Hbar @ taus[nu] - taus[nu] @ Hbar) @ phi
    bs = np.zeros((N, n))
    cs = np.zeros((N, n))
    onepl = np.eye(dim) + Lam
    for p in range(N):
        abar = emT @ a[p] @ eT
        adbar = emT @ ad[p] @ eT
        for mu in range(n):
            bs[p, mu] = phi @ taus[mu].T @ adbar @ phi
            cs[p, mu] = phi @ onepl @ abar @ taus[mu] @ phi
    return HEA, bs, cs
