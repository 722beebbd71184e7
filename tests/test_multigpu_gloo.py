"""The N > 1 host logic (sharding over spectra, max-over-ranks timing, candidate gathering) on CPU with gloo, world 2.
The search itself has no cross-rank data path: ranks are independent."""
import os
import sys
from pathlib import Path

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parents[1]


def _worker(rank, world, port, tmp):
    sys.path.insert(0, str(ROOT))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2406_15186_b200 import dist as pdist
    import oracle

    assert pdist.env_rank_world() == (rank, rank, world)
    # strong-scaling shard: contiguous, disjoint, complete
    batch = 5
    mine = pdist.shard_batch(batch, rank, world)
    # every rank searches its share with the (CPU) oracle standing in for the per-GPU plan
    rng = np.random.default_rng(123)
    specs = (rng.normal(0, 9, (batch, 3001)) + 1j * rng.normal(0, 9, (batch, 3001))).astype(np.complex64)
    specs[3, 700:712] *= 3
    specs[1, 100:104] *= 5
    local = oracle.search(specs[mine.start:mine.stop], 16, 512, 64, 3.5)
    local20 = np.zeros(len(local), dtype=[("spectrum", "<i4"), ("bin", "<i4"), ("width", "<i4"), ("power", "<f4"), ("sigma", "<f4")])
    for k in local20.dtype.names:
        local20[k] = local[k]
    parts = pdist.gather_candidates(local20, mine.start)
    merged = np.concatenate(parts)
    full = oracle.search(specs, 16, 512, 64, 3.5)
    assert np.array_equal(merged["spectrum"], full["spectrum"]) and np.array_equal(merged["bin"], full["bin"])
    assert np.array_equal(merged["width"], full["width"])
    # timing reduction: max over ranks; units: sum over ranks
    assert pdist.max_over_ranks(1.0 + rank) == float(world)
    assert pdist.sum_over_ranks(10.0) == 10.0 * world
    pdist.barrier()
    Path(tmp, f"ok{rank}").write_text("ok")
    dist.destroy_process_group()


def test_two_ranks_gloo(tmp_path):
    import oracle
    oracle.build()
    port = 29600 + os.getpid() % 1000
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    assert (tmp_path / "ok0").exists() and (tmp_path / "ok1").exists()


def test_shard_batch_partitions():
    sys.path.insert(0, str(ROOT))
    from paper_2406_15186_b200 import dist as pdist
    for batch in (1, 7, 256, 2048):
        for world in (1, 2, 3, 8):
            parts = [pdist.shard_batch(batch, r, world) for r in range(world)]
            assert [i for p in parts for i in p] == list(range(batch))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
