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


def _bench(*argv, env=None):
    import json
    import subprocess
    e = dict(os.environ)
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT"):
        e.pop(k, None)
    e.update(env or {})
    res = subprocess.run([sys.executable, str(ROOT / "bench.py"), *argv], capture_output=True, text=True, env=e, timeout=300)
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    return res, (json.loads(lines[-1]) if lines else None)


@pytest.mark.parametrize("scaling", ["strong", "weak"])
def test_bench_launches_its_own_ranks_at_world_size_2(scaling):
    """`python bench.py --gpus 2` outside torchrun must start 2 ranks by itself (bench.self_launch); --launch-check runs the
    launcher, the rank environment, the shard assignment and the MAX reduction on gloo without touching a GPU."""
    res, line = _bench("--launch-check", "--gpus", "2", "--scaling", scaling, "--config", "4")
    assert res.returncode == 0, res.stderr[-2000:]
    assert line["launch_check"] and line["n_gpus"] == 2 and line["scaling"] == scaling
    ranks = sorted(line["ranks"])
    assert [r[0] for r in ranks] == [0, 1] and [r[1] for r in ranks] == [0, 1]          # rank, local rank
    nx = line["nx"]
    assert nx == 32 ** 3
    if scaling == "strong":                          # config 4's 32 768 cells split in two contiguous halves
        assert [tuple(r[2:]) for r in ranks] == [(0, nx // 2), (nx // 2, nx)]
    else:                                            # one copy per rank at distinct global offsets
        assert [tuple(r[2:]) for r in ranks] == [(0, nx), (nx, 2 * nx)]
    assert line["max_over_ranks"] == 2.0
    assert line["nccl_debug"] == "INFO"              # set by the launcher unless the caller chose otherwise


def test_bench_refuses_a_world_size_that_contradicts_gpus():
    res, line = _bench("--launch-check", "--gpus", "2", env=dict(RANK="0", WORLD_SIZE="4", LOCAL_RANK="0"))
    assert res.returncode != 0 and "WORLD_SIZE=4" in res.stderr and line is None


@pytest.mark.skipif(__import__("torch").cuda.is_available(), reason="checks the too-few-GPUs failure mode on a box without GPUs")
def test_bench_refuses_to_run_fewer_ranks_than_asked_for():
    res, line = _bench("--gpus", "2")
    assert res.returncode != 0 and "only 0 CUDA device" in res.stderr and line is None


def test_workload_shards_concatenate_to_the_unsharded_input():
    """bench.py's strong-scaling ranks build only their own cells (workloads.make(cells=...)): same bits as slicing."""
    import workloads
    from paper_2308_04869_b200 import sharding
    for cfg, kw in ((2, dict(nx=7, np_side=4)), (4, dict(nx=9, np_side=4)), (3, dict(nx=5, np_side=4)), (7, dict(nx=4, np_side=3))):
        w = workloads.make(cfg, **kw)
        for world in (2, 3):
            for r in range(world):
                lo, hi = sharding.cell_range(w["problem"]["nx"], r, world)
                ws = workloads.make(cfg, cells=(lo, hi), **kw)
                _, fl, off = sharding.shard_problem(w["problem"], w["f"], r, world)
                assert off == lo == ws["ix_offset"] and ws["problem"]["nx"] == hi - lo and ws["nx_global"] == w["problem"]["nx"]
                assert np.array_equal(fl, ws["f"])
