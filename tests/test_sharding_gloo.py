"""Multi-GPU host logic on CPU: world_size-2 gloo process group.

Spatial cells are independent (Eq. 16 is local in x), so the N > 1 path is: each
rank owns a contiguous range of cells, computes them with the stream keyed by the GLOBAL cell
index, and nothing is exchanged except the MAX all-reduce of the timing.  There is no GPU here, so
the per-rank compute is played by the oracle (tests may use it); what is under test is the
product's host-side code: sharding.cell_range / shard_problem / unshard / max_over_ranks."""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, tmp):
    sys.path.insert(0, str(ROOT))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      OMP_NUM_THREADS="2")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        import workloads
        from paper_2308_04869_b200 import sharding
        w = workloads.make(2, nx=5, np_side=6, n_samples=40)
        prob, f = w["problem"], w["f"]
        local_prob, local_f, lo = sharding.shard_problem(prob, f, rank, world)
        hi = lo + local_prob["nx"]
        assert (lo, hi) == sharding.cell_range(5, rank, world)
        # per-rank compute on the local shard with the global cell offset: the oracle evaluates cells
        # [lo, hi) of the global problem, then the rank keeps only its own rows (= what rbg_collision
        # returns for a handle created with ix_offset = lo)
        orc = oracle.Oracle(prob)
        C_full_cells = orc.collision(f, w["n_samples"], w["seed"], ix_begin=lo, ix_end=hi)
        _, C_local, _ = sharding.shard_problem(prob, C_full_cells, rank, world)
        assert C_local.shape == local_f.shape
        np.save(Path(tmp) / f"C_{rank}.npy", C_local)
        # the only collective on the path: MAX of the per-rank step time
        t = sharding.max_over_ranks(1.0 + rank)
        assert t == float(world)
        dist.barrier()
        if rank == 0:
            pieces = [np.load(Path(tmp) / f"C_{r}.npy") for r in range(world)]
            whole = sharding.unshard(prob, pieces)
            ref = orc.collision(f, w["n_samples"], w["seed"])
            assert np.array_equal(whole, ref)
            assert np.any(ref != 0)
    finally:
        dist.destroy_process_group()


def test_world_size_2_sharding_reproduces_the_single_rank_result(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)


@pytest.mark.parametrize("nx,world", [(5, 2), (7, 3), (8, 8), (3, 4), (1, 2)])
def test_cell_ranges_partition_the_domain(nx, world):
    from paper_2308_04869_b200 import sharding
    seen = []
    for r in range(world):
        lo, hi = sharding.cell_range(nx, r, world)
        assert 0 <= lo <= hi <= nx
        seen.extend(range(lo, hi))
    assert seen == list(range(nx))
    sizes = [sharding.cell_range(nx, r, world)[1] - sharding.cell_range(nx, r, world)[0] for r in range(world)]
    assert max(sizes) - min(sizes) <= 1


def test_shard_unshard_roundtrip():
    import workloads
    from paper_2308_04869_b200 import sharding
    w = workloads.make(3, nx=7, np_side=4, n_samples=8)
    for world in (1, 2, 3):
        pieces = [sharding.shard_problem(w["problem"], w["f"], r, world)[1] for r in range(world)]
        assert np.array_equal(sharding.unshard(w["problem"], pieces), w["f"])
