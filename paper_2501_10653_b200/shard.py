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


# ----------------------------------------------------------------------------- one pair over several GPUs
def band_rows(H: int, N_T: int, rank: int, world: int) -> tuple:
    """Rows [r0, r1) of an H-row image that ``rank`` owns when ONE pair is sharded over ``world`` GPUs
    (SURVEY.md 8(e)): contiguous bands of whole tile rows (a band is one contiguous byte range of a
    row-major image, no halo), balanced to within one tile row; the last band takes the ragged rest."""
    if world <= 0 or not 0 <= rank < world or H <= 0 or N_T <= 0:
        raise ValueError("bad (H, N_T, rank, world)")
    nty = -(-H // N_T)
    tr = pair_range(nty, rank, world)                    # tile rows of this rank
    return min(H, tr.start * N_T), min(H, tr.stop * N_T)


def banded_pair(binding, x_band, y_band, n_tiles_total: int, N_T: int, C1, C2, C, D, dist=None) -> dict:
    """One rank's share of ONE image pair sharded by bands of tile rows: Eqs. 1-2 for the tiles of the band
    (``iqa_fused_tiles_2d``; no exchange), then the whole-image pair of Eqs. 3-4 through ONE all-reduce of
    four doubles (``iqa_aggregate_partial`` -> ``dist.all_reduce`` -> ``iqa_aggregate_finish``).
    x_band, y_band: this rank's rows (CUDA tensors, possibly empty when there are more ranks than tile
    rows).  Returns the band's matrices plus ``whole`` = [LISI, augLISI] of the ENTIRE image on every rank."""
    import torch
    dev = x_band.device
    if x_band.shape[0] > 0:
        out = binding.fused_tiles_2d(x_band, y_band, N_T, C1, C2, C, D)
        sums4 = binding.aggregate_partial(out["lisi"], out["auglisi"], out["X"], out["Y"], C2, C)
    else:
        out = {k: torch.empty((0, -(-x_band.shape[1] // N_T)), dtype=torch.float32, device=dev)
               for k in ("lisi", "auglisi", "X", "Y")}
        sums4 = torch.zeros(4, dtype=torch.float64, device=dev)
    sums4 = allreduce_sums(sums4, dist)
    out["whole"] = binding.aggregate_finish(sums4, n_tiles_total, C2, C)
    return out


def allreduce_sums(sums4, dist=None):
    """Sum of the per-band partial sums of Eqs. 3-4 over all ranks (32 bytes; the path's only exchange)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return sums4
    dist.all_reduce(sums4, op=dist.ReduceOp.SUM)
    return sums4
