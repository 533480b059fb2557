"""Shared test helpers: random tiny systems in the C-ABI layouts (numpy), packing helpers."""
import numpy as np


def antisym4(x):
    x = x - x.transpose(1, 0, 2, 3)
    return x - x.transpose(0, 1, 3, 2)


def pack_pairs(t2):
    """full [o,o,v,v] -> pair-packed [npair,v,v]"""
    o = t2.shape[0]
    iu = np.triu_indices(o, 1)
    return np.ascontiguousarray(t2[iu[0], iu[1]])


def pack_full(t2):
    """full [o,o,v,v] -> [npair, ntri]"""
    o, v = t2.shape[0], t2.shape[2]
    iu = np.triu_indices(o, 1)
    au = np.triu_indices(v, 1)
    return np.ascontiguousarray(t2[iu[0], iu[1]][:, au[0], au[1]])


def random_system(o, v, Q, seed, sym_L=True, diag_f=False, t_scale=0.1, l_scale=0.3):
    rng = np.random.default_rng(seed)
    N = o + v
    L = rng.normal(size=(Q, N, N)) * l_scale
    if sym_L:
        L = 0.5 * (L + L.transpose(0, 2, 1))
    f = rng.normal(size=(N, N)) * 0.2
    f = 0.5 * (f + f.T) + np.diag(np.concatenate([-1 - rng.random(o), 0.5 + rng.random(v)]))
    if diag_f:
        f = np.diag(np.diag(f))
    t1 = rng.normal(size=(o, v)) * t_scale
    l1 = rng.normal(size=(o, v)) * t_scale
    t2 = antisym4(rng.normal(size=(o, o, v, v)) * t_scale)
    l2 = antisym4(rng.normal(size=(o, o, v, v)) * t_scale)
    return dict(o=o, v=v, Q=Q, fock=f, Lchol=np.ascontiguousarray(L), T1=t1, L1=l1, t2=t2, l2=l2,
                T2p=pack_pairs(t2), L2p=pack_full(l2))


def random_x(o, v, nrhs, seed):
    rng = np.random.default_rng(seed)
    x1 = rng.normal(size=(nrhs, o)) + 1j * rng.normal(size=(nrhs, o))
    x2 = rng.normal(size=(nrhs, o, o, v)) + 1j * rng.normal(size=(nrhs, o, o, v))
    x2 = x2 - x2.transpose(0, 2, 1, 3)
    return x1, x2


def relmax(a, b):
    a = np.asarray(a)
    b = np.asarray(b)
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


def to_numpy_system(s):
    """gfcc_inputs dict of torch tensors -> dict of numpy arrays (host)."""
    out = {}
    for k, val in s.items():
        out[k] = val.cpu().numpy() if hasattr(val, "cpu") else val
    return out
