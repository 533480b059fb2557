"""Closed-shell (spin-restricted) inputs for the oracle -- TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

The paper ran a spin-explicit closed-shell code that "only deals with the alpha electrons" (Table 2 note).  For a
closed-shell reference the spin-free amplitudes define the spin-orbital ones, and the closed-shell Green's function IS the
spin-orbital one on the expanded tensors (alpha targets).  This module writes that expansion out; the oracle proper (oracle.Oracle)
then runs unchanged.  Spin-free definition (pinned in tests/test_oracle_closed_shell.py by a Fock-space brute force built from the
spin-summed excitation operators E_pq = sum_s a+_ps a_qs):
    T = sum_ia t1[i,a] E_ai + 1/2 sum_ijab t2[i,j,a,b] E_ai E_bj,      t2[i,j,a,b] = t2[j,i,b,a]   (same form for Lambda)
    spin-orbital:  t[is, jt, as', bt'] = d(s,s') d(t,t') t2[i,j,a,b] - d(s,t') d(t,s') t2[i,j,b,a];   t[is, as'] = d(s,s') t1[i,a]
    f[ps, qs'] = d(s,s') f[p,q];   L[Q, ps, qs'] = d(s,s') L[Q,p,q]
Spin-orbital ordering ("blocked"): occupied alpha (no), occupied beta (no), virtual alpha (nv), virtual beta (nv).
"""
import numpy as np


def so_index(no, nv, p, spin):
    """spin-orbital index of spatial orbital p (0..no+nv-1) with spin 0 (alpha) / 1 (beta)"""
    return spin * no + p if p < no else 2 * no + spin * nv + (p - no)


def _doubles(no, nv, x):
    o, v = 2 * no, 2 * nv
    t = np.zeros((o, o, v, v))
    for s in range(2):
        for u in range(2):
            I, J = slice(s * no, (s + 1) * no), slice(u * no, (u + 1) * no)
            A, B = slice(s * nv, (s + 1) * nv), slice(u * nv, (u + 1) * nv)
            t[I, J, A, B] += x
            t[I, J, B, A] -= x.transpose(0, 1, 3, 2)
    return t


def expand_closed_shell(no, nv, fock_s, T1_s, T2_s, L1_s, L2_s, Lchol_s):
    """spatial tensors (fock [Ns,Ns], T1/L1 [no,nv], T2/L2 [no,no,nv,nv], Lchol [Q,Ns,Ns]) -> dict of spin-orbital tensors in the
    C-ABI layouts of include/gfcc.h (o = 2 no, v = 2 nv): fock, T1, T2p, L1, L2p, Lchol, plus the full t2, l2."""
    Ns, o, v = no + nv, 2 * no, 2 * nv
    N = o + v
    Q = Lchol_s.shape[0]
    f = np.zeros((N, N))
    L = np.zeros((Q, N, N))
    for s in range(2):
        idx = [so_index(no, nv, p, s) for p in range(Ns)]
        f[np.ix_(idx, idx)] = fock_s
        for q in range(Q):
            L[q][np.ix_(idx, idx)] = Lchol_s[q]
    t1 = np.zeros((o, v))
    l1 = np.zeros((o, v))
    for s in range(2):
        t1[s * no:(s + 1) * no, s * nv:(s + 1) * nv] = T1_s
        l1[s * no:(s + 1) * no, s * nv:(s + 1) * nv] = L1_s
    t2, l2 = _doubles(no, nv, np.asarray(T2_s)), _doubles(no, nv, np.asarray(L2_s))
    iu, au = np.triu_indices(o, 1), np.triu_indices(v, 1)
    return dict(o=o, v=v, Q=Q, fock=f, Lchol=L, T1=t1, L1=l1, t2=t2, l2=l2,
                T2p=np.ascontiguousarray(t2[iu[0], iu[1]]), L2p=np.ascontiguousarray(l2[iu[0], iu[1]][:, au[0], au[1]]))
