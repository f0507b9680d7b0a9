"""Host-side sharding of the path across GPUs (one process per GPU).

The (field, scale) right-hand sides are independent solves on a read-only prepared mesh, so the path shards
over right-hand sides with no data-path collective: every rank keeps its own replica of the mesh and solves its
own fields.  Only timings / small result tables are gathered (torch.distributed, NCCL on GPUs, gloo in the CPU
tests).  No arithmetic of the method lives here.
"""
from __future__ import annotations

from typing import List, Sequence, Tuple


def rank_fields(n_fields: int, world: int, rank: int) -> slice:
    """Contiguous, balanced slice of the fields owned by `rank` (sizes differ by at most one)."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad world/rank")
    base, extra = divmod(n_fields, world)
    start = rank * base + min(rank, extra)
    return slice(start, start + base + (1 if rank < extra else 0))


def partition_rhs(ells: Sequence[float], n_fields: int, order_n: int, world: int) -> List[List[Tuple[int, int]]]:
    """Strong-scaling split of ONE job: (field, scale) pairs distributed by estimated cost (iterations grow like
    l^n), longest-processing-time first, so that ranks finish together.  Returns per rank a list of (f, j)."""
    cost = [float(l) ** order_n for l in ells]
    items = sorted(((cost[j], f, j) for f in range(n_fields) for j in range(len(ells))), reverse=True)
    load = [0.0] * world
    out: List[List[Tuple[int, int]]] = [[] for _ in range(world)]
    for c, f, j in items:
        r = min(range(world), key=lambda i: (load[i], i))
        out[r].append((f, j))
        load[r] += c
    for lst in out:
        lst.sort()
    return out


def gather_max(value: float, group=None) -> float:
    """Max over ranks of a host scalar (timings)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    t = torch.tensor([value], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def gather_table(local_rows, group=None):
    """All ranks' small result tables (lists of picklable rows) concatenated in rank order."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return list(local_rows)
    world = dist.get_world_size(group)
    out = [None] * world
    dist.all_gather_object(out, list(local_rows), group=group)
    return [row for part in out for row in part]
