"""Pin of the closed-shell (spin-restricted) expansion used for PAPER.md:244's closed-shell workflow (oracle/closed_shell.py)
against the SPIN-FREE definition on Fock space: H, T and Lambda written with the spin-summed excitation operators
E_pq = sum_s a+_ps a_qs and spatial integrals / amplitudes only -- independent of any spin-orbital expansion formula."""
import numpy as np
import pytest
from scipy.linalg import expm

import oracle
from oracle.closed_shell import expand_closed_shell, so_index
import gfcc_fockspace as fs


def spatial_system(no, nv, Q, seed):
    rng = np.random.default_rng(seed)
    Ns = no + nv
    L = rng.normal(size=(Q, Ns, Ns)) * 0.3
    L = 0.5 * (L + L.transpose(0, 2, 1))
    f = rng.normal(size=(Ns, Ns)) * 0.2
    f = 0.5 * (f + f.T) + np.diag(np.concatenate([-1 - rng.random(no), 0.5 + rng.random(nv)]))
    sym = lambda x: 0.5 * (x + x.transpose(1, 0, 3, 2))
    return dict(no=no, nv=nv, Q=Q, fock=f, Lchol=L, T1=rng.normal(size=(no, nv)) * 0.1, L1=rng.normal(size=(no, nv)) * 0.1,
                T2=sym(rng.normal(size=(no, no, nv, nv)) * 0.1), L2=sym(rng.normal(size=(no, no, nv, nv)) * 0.1))


def spinfree_operators(s):
    """H_N, T, Lambda as 2^N x 2^N matrices from the spin-free definitions (blocked spin-orbital ordering for the JW strings)"""
    no, nv = s["no"], s["nv"]
    Ns, o, v = no + nv, 2 * no, 2 * nv
    N = o + v
    a = fs.jw_annihilators(N)
    ad = [x.T for x in a]
    dim = 2 ** N
    E = [[sum(ad[so_index(no, nv, p, sp)] @ a[so_index(no, nv, q, sp)] for sp in range(2)) for q in range(Ns)] for p in range(Ns)]
    g = np.einsum("Qpr,Qqs->pqrs", s["Lchol"], s["Lchol"])                 # <pq|rs>
    h = s["fock"] - 2 * np.einsum("pkqk->pq", g[:, :no, :, :no]) + np.einsum("pkkq->pq", g[:, :no, :no, :])
    H = np.zeros((dim, dim))
    for p in range(Ns):
        for q in range(Ns):
            H += h[p, q] * E[p][q]
            for r in range(Ns):
                for t in range(Ns):
                    H += 0.5 * g[p, q, r, t] * (E[p][r] @ E[q][t] - (E[p][t] if q == r else 0.0))
    phi = np.zeros(dim)
    phi[0] = 1.0
    for p in reversed(range(o)):
        phi = ad[p] @ phi
    HN = H - (phi @ H @ phi) * np.eye(dim)
    T = np.zeros((dim, dim))
    Lam = np.zeros((dim, dim))
    for i in range(no):
        for aa in range(nv):
            T += s["T1"][i, aa] * E[no + aa][i]
            Lam += s["L1"][i, aa] * E[i][no + aa]
            for j in range(no):
                for bb in range(nv):
                    T += 0.5 * s["T2"][i, j, aa, bb] * E[no + aa][i] @ E[no + bb][j]
                    Lam += 0.5 * s["L2"][i, j, aa, bb] * E[i][no + aa] @ E[j][no + bb]
    return a, ad, phi, HN, T, Lam


@pytest.mark.parametrize("no,nv", [(1, 2), (2, 1), (2, 2)])
def test_expansion_equals_spinfree_definition(no, nv):
    s = spatial_system(no, nv, 3, seed=10 * no + nv)
    x = expand_closed_shell(no, nv, s["fock"], s["T1"], s["T2"], s["L1"], s["L2"], s["Lchol"])
    o, v = x["o"], x["v"]
    a, ad, phi, HN, T, Lam = spinfree_operators(s)
    ops = fs.operators(o, v, x["fock"], x["Lchol"], x["T1"], x["t2"], x["L1"], x["l2"])
    Hbar_sf = expm(-T) @ HN @ expm(T)
    assert np.abs(Hbar_sf - ops[3]).max() < 1e-12                        # Hbar: f, L, T1, T2 expansion
    assert np.abs(Lam - ops[4]).max() < 1e-14                            # Lambda1, Lambda2 expansion
    # G for alpha targets through the oracle on the expanded tensors = literal definition with the spin-free operators
    orc = oracle.Oracle(o, v, x["Q"], x["fock"], x["T1"], x["T2p"], x["L1"], x["L2p"], x["Lchol"], oracle.MODE_DEF | oracle.MODE_EA)
    HIP, bs, cs = fs.brute_force(o, v, x["fock"], x["Lchol"], x["T1"], x["t2"], x["L1"], x["l2"], (a, ad, phi, Hbar_sf, Lam, expm(-T), expm(T)))
    targets = [so_index(no, nv, p, 0) for p in range(no + nv)]            # every spatial orbital, alpha spin
    w, eta = -0.41, 0.03
    n = HIP.shape[0]
    X = np.linalg.solve(HIP + (w - 1j * eta) * np.eye(n), bs[targets].T)
    Gref = (cs[targets] @ X).T
    G = orc.G_dense(targets, [w], eta)[0]
    assert np.abs(G - Gref).max() < 1e-11 * max(1.0, np.abs(Gref).max())
    # spin symmetry of the closed shell: G_{p alpha, q alpha} = G_{p beta, q beta}, G_{p alpha, q beta} = 0
    tb = [so_index(no, nv, p, 1) for p in range(no + nv)]
    Gall = orc.G_dense(targets + tb, [w], eta)[0]
    k = len(targets)
    assert np.abs(Gall[:k, :k] - Gall[k:, k:]).max() < 1e-11 * max(1.0, np.abs(Gall).max())
    assert np.abs(Gall[:k, k:]).max() < 1e-12 * max(1.0, np.abs(Gall).max())
