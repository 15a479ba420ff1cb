"""Host-side logic of the multi-GPU path: one process per GPU,
instances sharded by rank, NO collective on the data path (instances are independent, P:L87:
every instance has its own budget M).  Collectives only carry the report: the max over ranks of
the device time, the sum of the work counters and, when asked, the per-instance results.

Works with any ``torch.distributed`` backend (``nccl`` on the GPU box, ``gloo`` in the CPU
tests); holds none of the method's arithmetic.
"""
from __future__ import annotations

from typing import Sequence, Tuple

import torch
import torch.distributed as dist


def world() -> Tuple[int, int]:
    """(rank, world_size); (0, 1) without an initialised process group."""
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def weak_shard(rank: int, instances_per_rank: int) -> Tuple[int, int]:
    """Weak scaling (bench.py): rank r simulates the seeded instances
    [r * per_rank, (r + 1) * per_rank) -- per-GPU work is fixed as N grows."""
    if rank < 0 or instances_per_rank < 0:
        raise ValueError("rank and instances_per_rank must be >= 0")
    return rank * instances_per_rank, (rank + 1) * instances_per_rank


def strong_shard(n_instances: int, rank: int, world_size: int) -> Tuple[int, int]:
    """Strong scaling: contiguous balanced split of a fixed batch; the first ``n % world``
    ranks take one extra instance.  Ranges are disjoint and cover [0, n_instances)."""
    if not (0 <= rank < world_size) or n_instances < 0:
        raise ValueError("need 0 <= rank < world_size and n_instances >= 0")
    q, r = divmod(n_instances, world_size)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def reduce_report(times_ms: Sequence[float], counts: Sequence[float], device=None):
    """(max over ranks of every time, sum over ranks of every count) -- the contract of the
    bench line: device time is the slowest rank's, work is the whole job's."""
    rank, ws = world()
    t = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    c = torch.tensor(list(counts), dtype=torch.float64, device=device)
    if ws > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.tolist()], [float(x) for x in c.tolist()]


def gather_per_instance(local: torch.Tensor) -> torch.Tensor:
    """Concatenate the per-instance results of every rank in rank order (shards may differ in
    length).  One all_gather of the lengths and one of the padded values: 8 bytes per
    instance, latency-bound; off the timed path."""
    rank, ws = world()
    if ws == 1:
        return local.clone()
    n = torch.tensor([local.numel()], dtype=torch.int64, device=local.device)
    sizes = [torch.zeros_like(n) for _ in range(ws)]
    dist.all_gather(sizes, n)
    sizes = [int(s.item()) for s in sizes]
    cap = max(max(sizes), 1)
    pad = torch.zeros(cap, dtype=local.dtype, device=local.device)
    pad[: local.numel()] = local.reshape(-1)
    parts = [torch.zeros_like(pad) for _ in range(ws)]
    dist.all_gather(parts, pad)
    return torch.cat([p[:s] for p, s in zip(parts, sizes)])
