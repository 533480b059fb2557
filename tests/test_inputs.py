"""Seeded input generator: determinism, structure (symmetry / antisymmetry), element addressability."""
import numpy as np
import torch

import gfcc_inputs as gi


def test_hash_reference_values():
    # 32-bit mixing emulated in int64 must equal the same mixing done with python ints
    def mix(x):
        x ^= x >> 16; x = (x * 0x7FEB352D) & 0xFFFFFFFF
        x ^= x >> 15; x = (x * 0x846CA68B) & 0xFFFFFFFF
        x ^= x >> 16
        return x
    idx = torch.tensor([0, 1, 12345, 2**31 + 7, 2**32 - 1, 2**40 + 3], dtype=torch.int64)
    got = gi._hash(77, 3, idx).tolist()
    key = (77 * 0x9E3779B1 + 3 * 0x85EBCA77) & 0xFFFFFFFF
    want = [mix((int(i) & 0xFFFFFFFF) ^ mix((int(i) >> 32) ^ key)) for i in idx.tolist()]
    assert got == want


def test_uniform_normal_statistics():
    idx = torch.arange(400000, dtype=torch.int64)
    u = gi.uniform(5, 1, idx)
    assert 0.0 < float(u.min()) and float(u.max()) < 1.0
    assert abs(float(u.mean()) - 0.5) < 3e-3 and abs(float(u.var()) - 1 / 12) < 2e-3
    z = gi.normal(5, 2, idx)
    assert abs(float(z.mean())) < 6e-3 and abs(float(z.std()) - 1.0) < 6e-3
    assert abs(float((z ** 4).mean()) - 3.0) < 0.1


def test_structure_and_addressability():
    o, v, Q = 5, 7, 4
    s = gi.make_system(o, v, Q, seed=123)
    L = s["Lchol"]
    assert torch.equal(L, L.transpose(1, 2))
    T2p = s["T2p"]
    assert T2p.shape == (10, v, v) and torch.equal(T2p, -T2p.transpose(1, 2))
    # chunked generation gives the same bits as one-shot generation (element addressable)
    T2b = gi.doubles_pairpacked(o, v, 123, gi.TID_T2, chunk_pairs=3)
    assert torch.equal(T2p, T2b)
    # fully packed triangle of the same tensor id equals the a<b part of the pair-packed one
    Lp = gi.doubles_pairpacked(o, v, 123, gi.TID_L2)
    Lf = gi.doubles_fullpacked(o, v, 123, gi.TID_L2, chunk_pairs=4)
    iu = torch.triu_indices(v, v, 1)
    assert torch.equal(Lp[:, iu[0], iu[1]], Lf)
    # decay of the Cholesky vectors: rms of vector q ~ exp(-q/30)/sqrt(Q)
    L = gi.cholesky(20, 44, 60, seed=9)
    rms = L.pow(2).mean(dim=(1, 2)).sqrt()
    want = torch.exp(-torch.arange(60, dtype=torch.float64) / 30) / np.sqrt(60)
    assert float((rms / want - 1).abs().max()) < 0.08
    X1, X2 = gi.trial_vectors(o, v, 3, 123)
    assert torch.equal(X2, -X2.transpose(1, 2)) and X1.shape == (3, o)


def test_configs():
    c = gi.make_config(0)
    assert c["fock"].shape == (32, 32) and c["targets"] == [7, 6, 5, 4] and len(c["omegas"]) == 8
    assert float(c["omegas"][0]) == -1.0 and abs(float(c["omegas"][-1]) + 0.2) < 1e-15
    eo, ev = gi.orbital_energies(180, 660, gi.seed_of(4), banded=True)
    assert abs(float(eo.min()) + 1.002) < 1e-12 and abs(float(eo.max()) + 0.248) < 1e-12
    d = (eo[1:] - eo[:-1])
    assert int((d < 1.5e-3).sum()) == 36 * 4          # 36 five-fold near-degenerate groups
    assert float(ev.min()) >= 0.1 and float(ev.max()) <= 3.0
