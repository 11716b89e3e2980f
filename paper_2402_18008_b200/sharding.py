"""Multi-GPU plumbing: the path shards over independent homographies /
hypotheses with no data-path collective.  One process per GPU; each rank solves a contiguous
range.  The only exchange is RANSAC's final "best hypothesis" pick: an all-gather of
(count, global index, H) -- 48 bytes per rank, latency-only.

Host logic only (torch.distributed); no arithmetic of the method lives here.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_range(n: int, rank: int, world: int):
    """Contiguous [begin, end) of n independent units owned by `rank` of `world` ranks."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    base, rem = divmod(int(n), world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def combine_best(best_count: torch.Tensor, best_index_global: torch.Tensor, best_H: torch.Tensor, group=None):
    """Pick the winning hypothesis over all ranks: maximum count, ties -> lowest GLOBAL hypothesis index
    (reading R9).  Inputs are this rank's result: best_count int32 [1], best_index_global int64 [1]
    (local best index + the rank's shard offset; -1 with count -1 for an empty shard), best_H float32 [3,3].
    Works on CPU tensors (gloo) and CUDA tensors (NCCL).  Returns (count, index, H) identical on every rank."""
    world = dist.get_world_size(group)
    dev = best_count.device
    rec = torch.empty(11, dtype=torch.float64, device=dev)       # exact for int32 counts and indices < 2^53
    rec[0] = best_count.to(torch.float64).reshape(())
    rec[1] = best_index_global.to(torch.float64).reshape(())
    rec[2:] = best_H.reshape(9).to(torch.float64)
    out = [torch.empty_like(rec) for _ in range(world)]
    dist.all_gather(out, rec, group=group)
    allr = torch.stack(out)                                      # [world, 11]
    cnt, idx = allr[:, 0], allr[:, 1]
    valid = idx >= 0
    if not bool(valid.any()):
        return (torch.tensor([-1], dtype=torch.int32, device=dev), torch.tensor([-1], dtype=torch.int64, device=dev),
                torch.full((3, 3), float("nan"), dtype=torch.float32, device=dev))
    top = cnt[valid].max()
    cand = valid & (cnt == top)
    big = torch.full_like(idx, float(2 ** 62))
    w = int(torch.where(cand, idx, big).argmin())
    return (allr[w, 0:1].to(torch.int32), allr[w, 1:2].to(torch.int64), allr[w, 2:].to(torch.float32).reshape(3, 3))
