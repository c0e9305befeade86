"""Host-side multi-GPU plumbing.  Lines of sight are independent, so the path shards by
contiguous pixel ranges with the plan replicated and NO data-path collective; the only communication is
the timing reduction (max over ranks) and a barrier, both through torch.distributed."""
from __future__ import annotations


def shard_pixels(n_pix: int, rank: int, world: int, align: int = 128) -> tuple[int, int]:
    """[begin, end) of `rank`'s contiguous pixel range; interior boundaries fall on tile multiples."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    tiles = (n_pix + align - 1) // align
    lo = (tiles * rank) // world * align
    hi = (tiles * (rank + 1)) // world * align
    return min(lo, n_pix), min(hi, n_pix)


def rank_seed(seed: int, rank: int) -> int:
    """Weak scaling: every rank synthesises its own cube of the same shape."""
    return seed + 1000 * rank


def max_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: float, seconds_max: float, world: int) -> float:
    """Units all ranks processed / the slowest rank's time."""
    return world * units_per_rank / seconds_max
