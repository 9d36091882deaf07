"""Data-parallel plumbing of the operator over visibilities (Eq. 37-38): every rank
holds a replica of the image and its own visibilities; Phi needs no exchange, Phi^dagger ends with an
all-reduce(sum) of the n x n image.  On the CUDA path the exchange is issued from INSIDE the operator
(purify_grid_dist / purify_normal_dist hand the image to an all-reduce callback band by band, overlapped with the
crop - PurifyOp.normal_dist(x, out, allreduce=lambda band: dist.all_reduce(band))); this module holds what is left
for the host: the rank environment, who owns which visibilities, the timing rule.  torch.distributed only (NCCL on
GPUs, gloo in the CPU tests); no method arithmetic here and no import of oracle/ or of the CUDA library."""
from __future__ import annotations

import dataclasses
import os

import torch
import torch.distributed as dist


def world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process if absent)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def rank_config(cfg, rank: int):
    """Weak scaling: rank r draws its OWN visibility set - same recipe, seed offset by 100 r."""
    return cfg if rank == 0 else dataclasses.replace(cfg, index=cfg.index + 100 * rank)


def shard_bounds(M: int, rank: int, world_size: int):
    """Strong scaling helper: contiguous equal-count block [lo, hi) of M visibilities for `rank`
    (PAPER.md:307 'equal sections')."""
    base, extra = divmod(int(M), int(world_size))
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def allreduce_image(img: torch.Tensor) -> torch.Tensor:
    """Eq. (38): sum of the per-rank dirty images, in place.  Complex tensors go through their real view
    (gloo and NCCL both reduce real dtypes)."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(torch.view_as_real(img) if img.is_complex() else img, op=dist.ReduceOp.SUM)
    return img


def max_over_ranks(value: float, device=None) -> float:
    """Timing rule: a multi-rank number is the MAX over ranks."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        t = torch.tensor([float(value)], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())
    return float(value)


def barrier():
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()
