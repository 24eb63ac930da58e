"""Frequency sharding for N GPUs ("performed independently for each frequency").

The frequency lines are independent units; the only coupling is the imaging sum over frequencies
(PAPER.md:70).  Rank r of `world` migrates the lines `shard_lines(nw, r, world)` of the job with
its own plan (velocity and table replicated) and the partial images are summed with ONE
all-reduce -- the path's only exchange step.  No arithmetic of the method lives here.
"""
from __future__ import annotations

import numpy as np


def shard_lines(nw: int, rank: int, world: int) -> np.ndarray:
    """Indices of the frequency lines rank `rank` owns: round-robin, so every rank gets the same
    mix of low and high frequencies (table-slice size and work per line grow with frequency)."""
    if not (0 <= rank < world) or nw < 0:
        raise ValueError("bad rank/world/nw")
    return np.arange(rank, nw, world, dtype=np.int64)


def shard_workload(cfg: dict, rank: int, world: int) -> dict:
    """The rank's sub-workload: its omega lines and the matching rows of P0; everything else shared."""
    lines = shard_lines(cfg["nw"], rank, world)
    if lines.size == 0:
        raise ValueError("more ranks than frequency lines")
    out = dict(cfg)
    out["omega"] = np.ascontiguousarray(cfg["omega"][lines])
    out["P0"] = np.ascontiguousarray(cfg["P0"][lines])
    out["nw"] = int(lines.size)
    out["lines"] = lines
    return out


def allreduce_image(image, group=None):
    """image[z][x] = sum over ranks of the partial images (in place).  torch.distributed tensor
    (CUDA + nccl on the GPUs, CPU + gloo in the host-logic tests)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(image, op=dist.ReduceOp.SUM, group=group)
    return image
