"""Multi-GPU host logic: one process per GPU, SVD bins sharded across ranks, no data-path collective.

(bin, detector) pairs are independent units of work (groups of ~1000 templates are filtered
separately; one SVD bank per instrument).  Each rank builds a ``binding.Bank`` over
its own bins (``Bank(workload, precision, device, bins=shard)``), every rank is fed the same strain (8 KB per
detector-second), and only the compact triggers are gathered — with ``torch.distributed`` (nccl on GPUs, gloo in
the CPU tests).  Nothing here computes anything of the method: it partitions bin indices and moves trigger records.
"""
from __future__ import annotations

from typing import List, Sequence

import numpy as np


def bin_cost(bin_) -> float:
    """Tensor work per second of strain of one bin: sum_s L_s f_s (n_s + 2N) MACs (SURVEY.md §8(a) A2 + A3)."""
    rows = 2 * bin_.n_templates
    return float(sum(s.n_basis * s.rate * (s.n_taps + rows) for s in bin_.slices))


def shard_bins(costs: Sequence[float], world: int) -> List[List[int]]:
    """Longest-processing-time-first partition of bin indices over ``world`` ranks.  Deterministic (ties broken by
    bin index, then by rank), every bin appears exactly once, shards are returned sorted."""
    if world < 1:
        raise ValueError("world must be >= 1")
    order = sorted(range(len(costs)), key=lambda b: (-costs[b], b))
    load = [0.0] * world
    shards: List[List[int]] = [[] for _ in range(world)]
    for b in order:
        r = min(range(world), key=lambda i: (load[i], i))
        shards[r].append(b)
        load[r] += costs[b]
    return [sorted(s) for s in shards]


def to_global_bins(triggers: np.ndarray, shard: Sequence[int]) -> np.ndarray:
    """Rewrite the ``bin`` field of a rank's triggers (local index into its shard) to the global bin index."""
    out = triggers.copy()
    if len(out):
        out["bin"] = np.asarray(shard, dtype=np.int32)[out["bin"]]
    return out


def gather_triggers(local: np.ndarray, device=None, group=None) -> np.ndarray:
    """All-gather variable-length trigger arrays (32-byte records); every rank returns the concatenation in rank
    order.  ``device``: where the exchange buffers live ("cuda" for nccl, None/"cpu" for gloo)."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    n = torch.tensor([len(local)], dtype=torch.int64, device=device)
    counts = [torch.zeros(1, dtype=torch.int64, device=device) for _ in range(world)]
    dist.all_gather(counts, n, group=group)
    counts = [int(c.item()) for c in counts]
    cap = max(max(counts), 1)
    buf = torch.zeros(cap * local.dtype.itemsize, dtype=torch.uint8, device=device)
    if len(local):
        raw = torch.from_numpy(np.frombuffer(local.tobytes(), dtype=np.uint8).copy())
        buf[:raw.numel()] = raw.to(buf.device)
    bufs = [torch.zeros_like(buf) for _ in range(world)]
    dist.all_gather(bufs, buf, group=group)
    parts = [np.frombuffer(b.cpu().numpy().tobytes(), dtype=local.dtype)[:c] for b, c in zip(bufs, counts)]
    return np.concatenate(parts) if parts else local[:0]
