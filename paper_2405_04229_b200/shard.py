"""Multi-GPU plumbing: one process per GPU, segments sharded by contiguous id range.

The path shards with no data-path collective: every photon is a function of (seed, global segment
id, photon index) only, so a rank that is handed segments [lo, hi) with ``seg_id_base = lo``
produces exactly the photons the single-GPU run produces for those ids.  The one
exchange step is the final sum of the small per-rank results (ground histogram / camera histogram,
telescope counters, event counters), done with ``torch.distributed.all_reduce`` (NCCL over NVLink on
GPUs, gloo in the CPU tests); photon lists stay sharded.  With integral bunch weights the summed
histogram is bit-identical to the single-GPU one.
"""
from __future__ import annotations

from typing import Dict, List, Optional, Tuple


def plan_shards(n_segments: int, world_size: int) -> List[Tuple[int, int]]:
    """Contiguous, balanced [lo, hi) ranges covering 0..n_segments; empty ranges if world > n."""
    if n_segments < 0 or world_size < 1:
        raise ValueError("plan_shards: n_segments >= 0 and world_size >= 1 required")
    base, rem = divmod(n_segments, world_size)
    out, lo = [], 0
    for r in range(world_size):
        hi = lo + base + (1 if r < rem else 0)
        out.append((lo, hi))
        lo = hi
    return out


def shard_of(n_segments: int, rank: int, world_size: int) -> Tuple[int, int]:
    return plan_shards(n_segments, world_size)[rank]


def reduce_results(result: Dict[str, "object"], group=None, keys=("hist", "tel_counts", "counters")) -> Dict[str, "object"]:
    """In-place SUM all-reduce of the per-rank result tensors (hist, tel_counts, counters).

    ``counters[written]`` / ``overflow`` become job totals; each rank's photon list keeps its own
    length, returned as ``written_local``."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return result
    from .api import COUNTER_NAMES
    cnt = result.get("counters")
    if cnt is not None:
        result["written_local"] = int(cnt[COUNTER_NAMES.index("written")].item())
    for k in keys:
        t = result.get(k)
        if t is None:
            continue
        if not isinstance(t, torch.Tensor):
            raise TypeError(f"reduce_results: {k} must be a torch tensor")
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return result


def max_over_ranks(value: float, device: Optional[str] = None, group=None) -> float:
    """Max of a host scalar over the ranks (timing contract: a step takes as long as its slowest rank)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def sum_over_ranks(value: float, device: Optional[str] = None, group=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return float(t.item())
