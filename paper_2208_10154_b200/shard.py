"""Host-side logic of the multi-GPU (replica) mode: maps are independent units, so N ranks process disjoint blocks
of maps with no collective on the data path (the paper is single-GPU,
PAPER.md:251).  Only bookkeeping lives here: which global map indices a rank owns, and the max-over-ranks reduction
of a measured time.  No transform arithmetic."""
import numpy as np


def rank_map_indices(rank, world, nmaps_per_rank):
    """Global indices of the maps rank `rank` owns under weak scaling: a contiguous block of nmaps_per_rank."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    return np.arange(rank * nmaps_per_rank, (rank + 1) * nmaps_per_rank, dtype=np.int64)


def split_maps(nmaps_total, world):
    """Strong-scaling split of nmaps_total maps into `world` contiguous blocks whose sizes differ by at most one.
    Returns a list of (first, count)."""
    base, extra = divmod(nmaps_total, world)
    out, first = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((first, n))
        first += n
    return out


def max_over_ranks(value, device=None):
    """Max of a Python float over all ranks of the default process group (identity without a group)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
