"""Host-side task sharding of the GFCC (p, omega) list over ranks -- no arithmetic of the method lives here.

The paper's own parallelism is over independent (omega, p) tasks handed to process groups (Alg. 1
PAPER.md:209-224): every task is a separate linear system, so ranks never exchange data inside the solve loop.
One process per GPU; each rank owns a handle (the intermediates are replicated, "replication of
shared amplitudes") and solves its slice of the frequency grid; the only communication is the final gather of the
G matrices (np*np complex numbers per frequency -- control-path bytes, done with torch.distributed on whatever
backend the job runs: NCCL on GPUs, gloo in the CPU tests).
"""
import numpy as np


def omega_slice(n_total, world, rank):
    """[start, stop) of this rank's contiguous block of a frequency grid of n_total points; blocks differ by at most one
    point and cover the grid exactly (ranks beyond n_total get an empty block)."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("need world >= 1 and 0 <= rank < world")
    base, rem = divmod(int(n_total), world)
    start = rank * base + min(rank, rem)
    return start, start + base + (1 if rank < rem else 0)


def weak_scaling_grid(wlo, whi, nw_per_rank, world, rank):
    """bench.py's weak-scaling workload: the window [wlo, whi] sampled with nw_per_rank*world points, rank r solving the
    r-th block of nw_per_rank points (per-GPU work fixed as the job grows)."""
    grid = np.linspace(wlo, whi, nw_per_rank * world)
    a, b = omega_slice(len(grid), world, rank)
    return grid[a:b]


def gather_G(G_local, n_total, world, rank, dist=None, device="cpu"):
    """All-gather per-rank G blocks [nw_r, np, np] (complex128 numpy) into the full [n_total, np, np] array, ordered as the
    frequency grid.  dist: the torch.distributed module of an initialised job (None or world == 1: returns G_local)."""
    G_local = np.ascontiguousarray(G_local, dtype=np.complex128)
    if dist is None or world == 1:
        return G_local
    import torch
    npq = G_local.shape[1:]
    nmax = max(omega_slice(n_total, world, r)[1] - omega_slice(n_total, world, r)[0] for r in range(world))
    pad = np.zeros((nmax,) + npq, dtype=np.complex128)
    pad[:G_local.shape[0]] = G_local
    mine = torch.view_as_real(torch.from_numpy(pad)).contiguous().to(device)
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine)
    out = np.empty((n_total,) + npq, dtype=np.complex128)
    for r in range(world):
        a, b = omega_slice(n_total, world, r)
        out[a:b] = torch.view_as_complex(parts[r].cpu()).numpy()[:b - a]
    return out


def max_over_ranks(value, world, dist=None, device="cpu"):
    """device-time reduction used by bench.py: the step time of the job is the slowest rank's."""
    if dist is None or world == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
