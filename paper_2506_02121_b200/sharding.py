"""Multi-GPU host logic: the phase grid shards across ranks, nothing else.

Rows (phases) are independent given any seed, so rank r of W solves the contiguous rows
[r * n, (r + 1) * n) of a grid of W * n phases: it calls the library with num_phi = n and
mlcc_options.phi_index_offset = r * n, phi_index_total = W * n.  Stars are replicated (<= 1.2 MB);
there is no data-path collective.  The only collective is the max-reduce of the timings.
No arithmetic of the method lives here.
"""
from typing import List, Tuple


def phase_shard(rank: int, world: int, num_phi_per_rank: int) -> Tuple[int, int]:
    """-> (phi_index_offset, phi_index_total) of `rank` (weak scaling: every rank owns num_phi_per_rank rows)."""
    if world < 1 or not 0 <= rank < world or num_phi_per_rank < 1:
        raise ValueError("bad rank / world / num_phi_per_rank")
    return rank * num_phi_per_rank, world * num_phi_per_rank


def split_rows(num_phi_total: int, world: int) -> List[Tuple[int, int]]:
    """Strong-scaling split of a fixed grid: [(first_row, n_rows)] per rank, contiguous, sizes differ by <= 1."""
    if world < 1 or num_phi_total < world:
        raise ValueError("need at least one row per rank")
    out = []
    for r in range(world):
        a = (num_phi_total * r) // world
        b = (num_phi_total * (r + 1)) // world
        out.append((a, b - a))
    return out


def max_over_ranks(value: float, device=None) -> float:
    """Max of a per-rank scalar (the timing contract: a multi-GPU number is the slowest rank's)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
