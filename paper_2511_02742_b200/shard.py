"""Event sharding for the multi-GPU path: events are independent (PAPER.md L114-116 maps one window to one block), so
ranks take contiguous event ranges balanced by hit count and nothing is exchanged on the data path.

Host logic only (numpy + torch.distributed for the optional gather of per-event results); no Hough arithmetic here.
"""
from __future__ import annotations

from typing import List, Tuple

import numpy as np


def shard_events(offsets: np.ndarray, world_size: int) -> List[Tuple[int, int]]:
    """Contiguous event ranges [e0, e1) per rank with hit counts as equal as contiguous ranges allow.

    Cut k is placed at the event boundary whose cumulative hit count is nearest to k / world_size of the total (ties to
    the earlier boundary); with no hits at all the events themselves are split evenly.  Ranges cover 0..E exactly once,
    in rank order, and may be empty."""
    offsets = np.asarray(offsets, dtype=np.int64)
    n_events = len(offsets) - 1
    if world_size < 1 or n_events < 0:
        raise ValueError("world_size >= 1 and a valid offsets array are required")
    total = int(offsets[-1] - offsets[0]) if n_events else 0
    cuts = [0]
    for k in range(1, world_size):
        if total == 0:
            c = (n_events * k) // world_size
        else:
            target = offsets[0] + total * k / world_size
            c = int(np.searchsorted(offsets, target, side="left"))
            if c > 0 and abs(float(offsets[c - 1]) - target) <= abs(float(offsets[min(c, n_events)]) - target):
                c -= 1
            c = min(max(c, cuts[-1]), n_events)
        cuts.append(c)
    cuts.append(n_events)
    return [(cuts[r], cuts[r + 1]) for r in range(world_size)]


def local_batch(u: np.ndarray, v: np.ndarray, offsets: np.ndarray, rng: Tuple[int, int]):
    """(u, v, offsets) of the events [e0, e1) with offsets rebased to 0 (views where possible)."""
    e0, e1 = rng
    a, z = int(offsets[e0]), int(offsets[e1])
    return u[a:z], v[a:z], np.ascontiguousarray(offsets[e0:e1 + 1] - a)


def gather_per_event(local, ranges: List[Tuple[int, int]], group=None):
    """All-gather a per-event tensor (first dimension = local events) from every rank into event order.

    Returns the concatenation over ranks on every rank.  Uses torch.distributed (NCCL on GPUs, gloo on CPU); shards may
    have different lengths, so each is padded to the longest before the collective."""
    import torch
    import torch.distributed as dist

    world = dist.get_world_size(group)
    n_max = max(e1 - e0 for e0, e1 in ranges)
    pad = torch.zeros((n_max,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    return torch.cat([parts[r][: ranges[r][1] - ranges[r][0]] for r in range(world)], dim=0)
