"""Multi-process plumbing (one process per GPU): which slice of the tile work plan a rank takes, and the sum
of the ranks' integer histograms.  The pair count shards by work item with no data-path exchange (every rank
holds both catalogs, <= 80 MB); the only collective is this all-reduce of 3 x (nbins+2) 64-bit counters
(SURVEY.md 8(e)).  torch.distributed is the transport: NCCL for CUDA tensors, gloo for CPU tensors."""
from __future__ import annotations

import os
from typing import Tuple

import numpy as np
import torch
import torch.distributed as dist


def rank_world() -> Tuple[int, int]:
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def apply_partition(ctx) -> Tuple[int, int]:
    """Give this rank its share of the plan: work items w with w % world == rank (tpcf_set_partition)."""
    rank, world = rank_world()
    ctx.set_partition(rank, world)
    return rank, world


def allreduce_counts(counts):
    """Sum integer histograms over all ranks, in place for torch tensors; numpy arrays are returned summed.

    Counts are non-negative and < 2^63, so the uint64 histograms travel as int64 (NCCL and gloo both sum it).
    """
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return counts
    if isinstance(counts, np.ndarray):
        t = torch.from_numpy(counts.astype(np.int64, copy=True))
        if dist.get_backend() == "nccl":
            t = t.cuda()
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return t.cpu().numpy().astype(counts.dtype)
    dist.all_reduce(counts, op=dist.ReduceOp.SUM)
    return counts
