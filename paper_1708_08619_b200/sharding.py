"""Frame sharding over ranks: the paper's "split the trajectory, merge the results"
(PAPER.md:356, 727).  Frames are independent, so every rank accumulates its own
frames into its own plan and the uint64 count histograms are summed ONCE per run, before
g3_normalize.  No collective sits on the per-frame data path.  Host logic only (argument
marshalling around torch.distributed); works with any backend (nccl on GPUs, gloo in CPU tests).
"""
from __future__ import annotations

from typing import Tuple


def frame_shard(n_frames: int, rank: int, world: int) -> Tuple[int, int]:
    """[begin, end) of the contiguous block of frames rank `rank` of `world` processes;
    block sizes differ by at most one and the blocks tile [0, n_frames)."""
    if world < 1 or not 0 <= rank < world or n_frames < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(n_frames, world)
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def merge_counts(counts, group=None):
    """Sum the per-rank count histograms (int64 bit patterns of uint64; two's-complement
    addition is the same operation).  Returns a new tensor, identical on every rank."""
    import torch.distributed as dist
    out = counts.clone()
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(out, op=dist.ReduceOp.SUM, group=group)
    return out


def merge_frames(frames: int, device=None, group=None) -> int:
    """Total number of frames over all ranks."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([int(frames)], dtype=torch.int64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return int(t.item())
