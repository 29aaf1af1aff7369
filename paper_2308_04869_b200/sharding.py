"""Host-side spatial sharding for multi-GPU runs.

Eq. 16 couples only momenta at one (t, x), so spatial cells are independent
units: each rank owns a contiguous range of cells and there is NO data-path collective.  The sample
stream is keyed by the global cell index (``ix_offset``), so any partition reproduces the
single-device result bit for bit.
"""
from __future__ import annotations

import numpy as np


def cell_range(nx: int, rank: int, world: int):
    """Contiguous, balanced [lo, hi) range of spatial cells for ``rank`` of ``world``."""
    base, rem = divmod(nx, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def shard_problem(problem: dict, f: np.ndarray, rank: int, world: int):
    """Strong-scaling shard: (local_problem, local_f, ix_offset) of a global problem."""
    nx = int(problem["nx"])
    lo, hi = cell_range(nx, rank, world)
    parts, off = [], 0
    for g in problem["grids"]:
        npc = int(np.prod(g["n"]))
        parts.append(f[off:off + nx * npc].reshape(nx, npc)[lo:hi].reshape(-1))
        off += nx * npc
    return dict(problem, nx=hi - lo), np.concatenate(parts), lo


def unshard(problem: dict, pieces):
    """Inverse of shard_problem for a list of per-rank result arrays (rank order)."""
    nx = int(problem["nx"])
    world = len(pieces)
    out = []
    offs = [0] * world
    for g in problem["grids"]:
        npc = int(np.prod(g["n"]))
        for r in range(world):
            lo, hi = cell_range(nx, r, world)
            n = (hi - lo) * npc
            out.append(pieces[r][offs[r]:offs[r] + n])
            offs[r] += n
    return np.concatenate(out)


def max_over_ranks(value: float) -> float:
    """MAX all-reduce of a per-rank time (the multi-GPU timing rule); identity without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
