"""Host-side logic of the multi-GPU path.

The path shards by REPLICA WORD COLUMNS only: columns never interact (the
shifts Sigma, sigma_k do not depend on the word; everything else is keyed by the
global word index), so rank r runs an ordinary handle created with
word_offset = first column of its shard, and the union over ranks is
bit-identical to one big run.  There is no collective on the data path; the only
exchange is gathering the uint32 per-replica counts at record times (8 KiB at
R = 2048) and taking the max over ranks of the device time.  Backend-agnostic:
NCCL on GPUs, gloo in the CPU tests.
"""
from __future__ import annotations

import numpy as np


def shard_words(W: int, world_size: int, rank: int) -> tuple[int, int]:
    """Columns [w0, w1) owned by `rank`: contiguous, sizes differ by at most 1."""
    if not (0 <= rank < world_size):
        raise ValueError("rank out of range")
    base, extra = divmod(W, world_size)
    w0 = rank * base + min(rank, extra)
    return w0, w0 + base + (1 if rank < extra else 0)


def gather_counts(local_counts: np.ndarray, W: int, device=None) -> np.ndarray:
    """All ranks' per-replica counts in global replica order (uint32[64 W]).
    Shards may be ragged, so every rank pads to the largest shard."""
    import torch
    import torch.distributed as dist

    if not dist.is_initialized() or dist.get_world_size() == 1:
        return np.asarray(local_counts, dtype=np.uint32)
    world, rank = dist.get_world_size(), dist.get_rank()
    sizes = [64 * (b - a) for a, b in (shard_words(W, world, r) for r in range(world))]
    assert len(local_counts) == sizes[rank]
    pad = max(sizes)
    buf = torch.zeros(pad, dtype=torch.int64, device=device)
    buf[: sizes[rank]] = torch.from_numpy(np.asarray(local_counts).astype(np.int64)).to(buf.device)
    out = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(out, buf)
    return np.concatenate([o[:n].cpu().numpy() for o, n in zip(out, sizes)]).astype(np.uint32)


def max_over_ranks(value: float, device=None) -> float:
    """Max over ranks of a device-measured time (never wall clock)."""
    import torch
    import torch.distributed as dist

    if not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
