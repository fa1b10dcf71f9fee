"""Multi-GPU host logic: the search shards over the template bank (eq.11-12 partitions the
bank into sets W_alpha and runs independent GPUs, :211).  One process per GPU, each searches its own slice;
no collective on the data path.  The only exchange is the concatenation of the tail records on rank 0 after the
search: a host-side merge over a gloo group (the records are in pinned host memory already), exact sizes, no padding.
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


_host_groups: dict = {}


def _host_group(group):
    """A gloo group over the ranks of `group` (made once, collectively, on first use).  The records of a search are
    already in host memory when it returns, so they are merged on the host: no copy back to the device, no NCCL."""
    import torch.distributed as dist

    if dist.get_backend(group) == "gloo":
        return group
    key = id(group) if group is not None else None
    if key not in _host_groups:
        ranks = dist.get_process_group_ranks(group) if group is not None else None
        _host_groups[key] = dist.new_group(ranks=ranks, backend="gloo")
    return _host_groups[key]


def gather_tails(tails: np.ndarray, group=None, dst: int = 0):
    """Concatenate every rank's records on `dst` (returns None elsewhere), in rank order -- the host-side merge of the
    independent GPUs' outputs (PAPER.md:187-191 eq.17, :211).  Records are plain bytes (12 B each).  Sizes go first
    (one all_gather of an int64); then every rank with records sends exactly its own bytes to `dst` over gloo:
    nothing is padded to the largest rank and nothing passes through device memory.  Collective: every rank of
    `group` must call it.  `dst` is a global rank."""
    import torch
    import torch.distributed as dist

    pg = _host_group(group)
    rank = dist.get_rank()
    ranks = dist.get_process_group_ranks(pg) if pg is not None else list(range(dist.get_world_size()))
    raw = torch.from_numpy(np.ascontiguousarray(tails).view(np.uint8).reshape(-1).copy())
    counts = [torch.zeros(1, dtype=torch.int64) for _ in ranks]
    dist.all_gather(counts, torch.tensor([raw.numel()], dtype=torch.int64), group=pg)
    sizes = [int(c.item()) for c in counts]
    if rank != dst:
        if raw.numel():
            dist.send(raw, dst=dst, group=pg)
        return None
    parts = []
    for r, n in zip(ranks, sizes):
        if r == dst:
            parts.append(raw)
        elif n:
            buf = torch.empty(n, dtype=torch.uint8)
            dist.recv(buf, src=r, group=pg)
            parts.append(buf)
    return np.concatenate([b.numpy().view(tails.dtype) for b in parts]) if parts else tails[:0]
