"""N > 1 path on CPU: world_size-2 `gloo` job that shards the (p, omega) task list exactly as bench.py / a multi-GPU
user does (paper_2010_04768_b200.sharding), solves each rank's slice, gathers G and compares with the unsharded
result.  The per-rank "solver" here is the CPU oracle's dense-LU G (the GPU solver is covered by -m gpu parity);
what is under test is the host logic: slices cover the grid once, order is preserved, gather and max-reduction work."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2010_04768_b200 import sharding
from gfcc_testutil import random_system


def test_omega_slices_cover_grid_once():
    for n in (1, 2, 7, 16, 60, 64):
        for world in (1, 2, 3, 4, 8):
            seen = []
            for r in range(world):
                a, b = sharding.omega_slice(n, world, r)
                assert 0 <= a <= b <= n
                seen += list(range(a, b))
            assert seen == list(range(n))
            sizes = [sharding.omega_slice(n, world, r)[1] - sharding.omega_slice(n, world, r)[0] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.omega_slice(4, 2, 2)


def test_weak_scaling_grid_is_a_partition_of_the_window():
    full = np.linspace(-1.0, -0.25, 4 * 3)
    got = np.concatenate([sharding.weak_scaling_grid(-1.0, -0.25, 4, 3, r) for r in range(3)])
    assert np.array_equal(got, full)
    assert np.array_equal(sharding.weak_scaling_grid(-1.0, -0.25, 4, 1, 0), np.linspace(-1.0, -0.25, 4))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, nw_total, out_dir):
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        s = random_system(3, 4, 5, seed=11, l_scale=0.2)
        orc = oracle.Oracle(s["o"], s["v"], s["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"])
        grid = np.linspace(-0.9, -0.2, nw_total)
        a, b = sharding.omega_slice(nw_total, world, rank)
        plist = [2, 1]
        G_local = orc.G_dense(plist, grid[a:b], 0.02) if b > a else np.zeros((0, 2, 2), dtype=np.complex128)
        G = sharding.gather_G(G_local, nw_total, world, rank, dist)
        tmax = sharding.max_over_ranks(10.0 + rank, world, dist)
        np.save(os.path.join(out_dir, f"G{rank}.npy"), G)
        np.save(os.path.join(out_dir, f"t{rank}.npy"), np.array([tmax]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("nw_total", [5, 8])
def test_two_rank_gloo_sharded_G_equals_unsharded(tmp_path, nw_total):
    import oracle
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), nw_total, str(tmp_path)), nprocs=world, join=True)
    s = random_system(3, 4, 5, seed=11, l_scale=0.2)
    orc = oracle.Oracle(s["o"], s["v"], s["Q"], s["fock"], s["T1"], s["T2p"], s["L1"], s["L2p"], s["Lchol"])
    ref = orc.G_dense([2, 1], np.linspace(-0.9, -0.2, nw_total), 0.02)
    for r in range(world):
        G = np.load(tmp_path / f"G{r}.npy")
        assert G.shape == ref.shape
        assert np.array_equal(G, ref) or np.abs(G - ref).max() <= 1e-14 * np.abs(ref).max()
        assert np.load(tmp_path / f"t{r}.npy")[0] == 11.0
