"""Sharding by sample over ranks.

Systems never interact in the sweep or the refresh and q needs only the
replicas of one sample together, so the path shards by sample with NO
data-path collective.  Rank r owns `n_samples` samples starting at the global
sample index `r * stride`, stride = n_samples rounded up to a multiple of 32
(weak scaling); Philox counters use the global index, so every shard is
bit-identical to the same samples of one big run.  The only
communication is the gather of the per-system measurement rows and the
max-over-ranks of the device time.  Host-side plumbing only: no arithmetic of
the method lives here.
"""
from __future__ import annotations

import numpy as np


def sample_offset(rank: int, n_samples_per_rank: int) -> int:
    """Global index of the first sample of `rank`.  The library needs a multiple of 16, the sample block that shares
    the Philox calls of a refresh; the stride is rounded up to a multiple of 32 (a whole word of
    single-replica samples), which satisfies it."""
    if rank < 0 or n_samples_per_rank < 1:
        raise ValueError("rank must be >= 0 and n_samples_per_rank >= 1")
    stride = (int(n_samples_per_rank) + 31) // 32 * 32
    return int(rank) * stride


def max_over_ranks(x: float, device=None) -> float:
    """MAX all-reduce of a scalar (device time of the timed region)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_rows(local: np.ndarray, per_sample: int, device=None) -> np.ndarray:
    """Concatenate per-rank measurement rows [n_rows, n_local_samples*per_sample]
    (int64 sums of E, E_daemon or Q) along the system axis in rank order."""
    import torch
    import torch.distributed as dist
    local = np.ascontiguousarray(local, dtype=np.int64)
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local
    t = torch.from_numpy(local).to(device) if device is not None else torch.from_numpy(local)
    parts = [torch.empty_like(t) for _ in range(dist.get_world_size())]
    dist.all_gather(parts, t)
    return np.concatenate([p.cpu().numpy() for p in parts], axis=1)
