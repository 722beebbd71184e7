"""Multi-GPU plumbing: the search shards over spectra (beams / DM trials) with no data-path collective.

Every spectrum is independent ("~2000 beams", L534 "one DM-trial per CPU core"), so N ranks run N
independent plans on their own share of the batch.  The only cross-rank operations are host-side bookkeeping:
the max-over-ranks of the step time, the sum of the units processed, and (optionally) gathering the variable-length
candidate lists.  They work on any torch.distributed backend (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import os
from typing import List, Tuple

import numpy as np
import torch
import torch.distributed as dist


def env_rank_world() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when not launched by torchrun."""
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def shard_batch(batch: int, rank: int, world: int) -> range:
    """Contiguous share of `batch` spectra owned by `rank` (strong scaling: total work fixed)."""
    base, rem = divmod(batch, world)
    lo = rank * base + min(rank, rem)
    return range(lo, lo + base + (1 if rank < rem else 0))


def _device_for_backend() -> torch.device:
    return torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")


def max_over_ranks(value: float) -> float:
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=_device_for_backend())
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float) -> float:
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=_device_for_backend())
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def barrier() -> None:
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


def gather_candidates(local: np.ndarray, spectrum_offset: int) -> List[np.ndarray]:
    """All ranks' candidate records (structured arrays) with `spectrum` shifted to global indices; on every rank.

    A count all-gather followed by a padded all-gather of the records (a few KB): bandwidth is irrelevant.
    """
    rec = local.copy()
    rec["spectrum"] += spectrum_offset
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [rec]
    dev = _device_for_backend()
    world = dist.get_world_size()
    counts = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(world)]
    dist.all_gather(counts, torch.tensor([len(rec)], dtype=torch.int64, device=dev))
    nmax = max(int(c.item()) for c in counts)
    item = rec.dtype.itemsize
    buf = torch.zeros(max(1, nmax) * item, dtype=torch.uint8, device=dev)
    if len(rec):
        buf[: len(rec) * item] = torch.from_numpy(rec.view(np.uint8).copy()).to(dev)
    bufs = [torch.zeros_like(buf) for _ in range(world)]
    dist.all_gather(bufs, buf)
    return [b[: int(c.item()) * item].cpu().numpy().view(rec.dtype).copy() for b, c in zip(bufs, counts)]
