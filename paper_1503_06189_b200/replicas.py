"""Host-side helpers for running N independent replicas (one handle per GPU).  The path has no exchange step:
frequency channels are independent, so multi-GPU = disjoint channel ranges, results concatenate
along f.  Nothing here touches the data path; torch.distributed is used only for the timing barrier / max."""
from __future__ import annotations


def channel_ranges(n_freq: int, world_size: int) -> list[tuple[int, int]]:
    """Contiguous, balanced [begin, end) channel ranges, one per rank (earlier ranks take the remainder)."""
    if n_freq < 0 or world_size <= 0:
        raise ValueError("bad arguments")
    base, rem = divmod(n_freq, world_size)
    out, b = [], 0
    for r in range(world_size):
        e = b + base + (1 if r < rem else 0)
        out.append((b, e))
        b = e
    return out


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """Max of a per-rank scalar (elapsed time) over all ranks; identity when not distributed."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: float, world_size: int, seconds_max_over_ranks: float) -> float:
    """Whole-job throughput: units all ranks processed / the slowest rank's time (weak scaling)."""
    return units_per_rank * world_size / seconds_max_over_ranks
