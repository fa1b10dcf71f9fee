"""Multi-GPU host logic: the search shards over the template bank (eq.11-12 partitions the
bank into sets W_alpha and runs independent GPUs, :211).  One process per GPU, each searches its own slice;
no collective on the data path.  The only exchange is the concatenation of the (rare) tail records on
rank 0 after the search, done with torch.distributed (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import numpy as np


def shard_range(n_templates: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous, balanced slice [lo, hi) of the bank owned by `rank` (first `rem` ranks get one more)."""
    if not (0 <= rank < world) or n_templates < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n_templates, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def chunk_ranges(lo: int, hi: int, chunk: int):
    """Split [lo, hi) into pieces of at most `chunk` templates (bank chunks that fit HBM)."""
    if chunk <= 0:
        raise ValueError("chunk must be positive")
    return [(a, min(a + chunk, hi)) for a in range(lo, hi, chunk)]


def globalize(tails: np.ndarray, offset: int) -> np.ndarray:
    """Local template ids of a shard/chunk -> ids in the whole bank."""
    out = tails.copy()
    out["template_id"] += np.uint32(offset)
    return out


def gather_tails(tails: np.ndarray, group=None, dst: int = 0):
    """Concatenate every rank's records on `dst` (returns None elsewhere).  Records are plain bytes
    (12 B each); counts go first so that ranks with no tails cost nothing but the count."""
    import torch
    import torch.distributed as dist

    world, rank = dist.get_world_size(group), dist.get_rank(group)
    backend = dist.get_backend(group)
    dev = torch.device("cuda", torch.cuda.current_device()) if backend == "nccl" else torch.device("cpu")
    raw = torch.from_numpy(np.ascontiguousarray(tails).view(np.uint8).copy()).to(dev)
    counts = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(world)]
    dist.all_gather(counts, torch.tensor([raw.numel()], dtype=torch.int64, device=dev), group=group)
    sizes = [int(c.item()) for c in counts]
    width = max(max(sizes), 1)
    padded = torch.zeros(width, dtype=torch.uint8, device=dev)
    padded[: raw.numel()] = raw
    bufs = [torch.zeros(width, dtype=torch.uint8, device=dev) for _ in range(world)] if rank == dst else None
    dist.gather(padded, bufs, dst=dst, group=group)
    if rank != dst:
        return None
    parts = [b[:n].cpu().numpy().view(tails.dtype) for b, n in zip(bufs, sizes)]
    return np.concatenate(parts) if parts else tails[:0]
