"""Multi-GPU plumbing: the path shards over sky patches with no data-path collective.

PAPER.md L423 Eq. (45): the search cost is a plain product/sum over binary blocks, detectors, frequency bands and sky
patches -- the units are independent.  One process per GPU (torch.distributed); rank r of W owns the patches
{p : p mod W == r}; the band's peakgram is replicated.  The only exchange is result collection: per-patch toplists
(k x 24 bytes) gathered to rank 0, and the max-over-ranks of the device time for the benchmark.  No method arithmetic
lives here: the merge only orders records the kernels produced, by the same (statistic desc, index asc) rule (R-11).
"""
from __future__ import annotations

from typing import Dict, List, Optional

import numpy as np


def patches_of_rank(n_patches: int, rank: int, world: int) -> List[int]:
    """Round-robin partition of patch indices: rank r gets r, r + W, r + 2W, ..."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank / world size")
    return list(range(rank, n_patches, world))


def max_over_ranks(value: float, dist=None) -> float:
    """MAX all-reduce of a per-rank scalar (device time in ms); identity without a process group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, dist=None) -> float:
    """SUM all-reduce of a per-rank scalar (work units processed)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_toplists(local: Dict[int, np.ndarray], dist=None, dst: int = 0) -> Optional[Dict[int, np.ndarray]]:
    """Collect {patch index: toplist records} from every rank on rank `dst` (None elsewhere).  A patch index may be
    owned by one rank only."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return dict(local)
    world, rank = dist.get_world_size(), dist.get_rank()
    payload = {int(k): np.ascontiguousarray(v) for k, v in local.items()}
    out = [None] * world if rank == dst else None
    dist.gather_object(payload, out, dst=dst)
    if rank != dst:
        return None
    merged: Dict[int, np.ndarray] = {}
    for part in out:
        for k, v in part.items():
            if k in merged:
                raise ValueError(f"patch {k} reported by two ranks")
            merged[k] = v
    return merged


def merge_block_toplists(parts: List[np.ndarray], k: int, key: str = "count") -> np.ndarray:
    """Toplist of one patch whose binary grid was split into blocks processed by different ranks:
    the k best of the union by (statistic descending, template index ascending) -- indices must already be global."""
    if not parts:
        raise ValueError("no toplists to merge")
    allr = np.concatenate(parts)
    order = np.lexsort((allr["index"], -allr[key].astype(np.float64)))
    return allr[order[:k]]
