"""Host-side logic of the multi-GPU path: image pairs are independent
(tiles -- and a fortiori pairs -- are processed independently), so a job of
many pairs shards over ranks with NO data-path collective.  One process per GPU; the only
communication is the barrier / max-over-ranks of the timing and, if wanted, gathering the
per-pair whole-image indices (2 floats per pair) on rank 0.

Nothing here touches CUDA or the method's arithmetic, so it is covered by world_size-2
``gloo`` tests on CPU (tests/test_shard_gloo.py).
"""
from __future__ import annotations


def pair_range(n_pairs_total: int, rank: int, world: int) -> range:
    """Contiguous, balanced slice of a job of ``n_pairs_total`` pairs for ``rank`` (strong
    scaling: the first ``n_pairs_total % world`` ranks take one extra pair)."""
    if world <= 0 or not 0 <= rank < world or n_pairs_total < 0:
        raise ValueError("bad (n_pairs_total, rank, world)")
    base, extra = divmod(n_pairs_total, world)
    start = rank * base + min(rank, extra)
    return range(start, start + base + (1 if rank < extra else 0))


def weak_seeds(pairs_per_rank: int, rank: int, world: int, seed0: int = 0) -> list:
    """Weak scaling (what bench.py runs): every rank draws its own ``pairs_per_rank`` distinct
    synthetic pairs; seeds never collide across ranks."""
    if world <= 0 or not 0 <= rank < world or pairs_per_rank < 0:
        raise ValueError("bad (pairs_per_rank, rank, world)")
    return [seed0 + rank * pairs_per_rank + i for i in range(pairs_per_rank)]


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """Max of a per-rank scalar (elapsed ms) over all ranks; identity when not distributed."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank: int, elapsed_ms_local: float, dist=None, device="cpu") -> dict:
    """Whole-job numbers from per-rank ones: all ranks' units divided by the slowest rank's time."""
    world = 1 if dist is None or not dist.is_initialized() else dist.get_world_size()
    ms = max_over_ranks(elapsed_ms_local, dist, device)
    total = units_per_rank * world
    return {"world": world, "ms": ms, "units": total,
            "us_per_unit": ms * 1e3 / total if total else float("nan"),
            "units_per_s": total / (ms * 1e-3) if ms > 0 else float("inf")}


def gather_whole(whole_local, dist=None):
    """Collect the per-pair [LISI, augLISI] rows of every rank on all ranks, in rank order
    (result collection only -- 8 bytes per pair)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return whole_local
    import torch
    parts = [torch.empty_like(whole_local) for _ in range(dist.get_world_size())]
    dist.all_gather(parts, whole_local.contiguous())
    return torch.cat(parts, dim=0)
