"""Multi-GPU host logic: the phase grid shards across ranks, nothing else.

Rows (phases) are independent given any seed, so rank r of W solves the contiguous rows
[r * n, (r + 1) * n) of a grid of W * n phases: it calls the library with num_phi = n and
mlcc_options.phi_index_offset = r * n, phi_index_total = W * n.  Stars are replicated (<= 1.2 MB);
the solve has no data-path collective.  The only collectives are the max-reduce of the timings and, for the
post-processing that needs the whole closed curve (chain joining; the crossing map),
the two small exchanges of the SEAM: every rank receives the first row of the next rank (ring, the last rank gets
row 0 of the first: the curve closes), links its own last row to it with the library's own mlcc_link_rows, adds the
segments of its rows (the seam segment included) into a map of its own with mlcc_crossing_map(closed = 0), and the
integer maps are summed (one all-reduce): every segment of the closed polygons is counted by exactly one rank.
No arithmetic of the method lives here: `api` is the binding (paper_2506_02121_b200.api) or anything with the same
call signatures.
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


def solve_shard(api, star_xy, masses, kappa_s, gamma, num_phi_per_rank, tol, max_iter, rank, world, **opt_kwargs):
    """This rank's rows of the grid of world * num_phi_per_rank phases through the fused C-ABI call
    (mlcc_curves_and_caustics with phi_index_offset / phi_index_total).  -> (roots, caustics, Stats)."""
    off, total = phase_shard(rank, world, num_phi_per_rank)
    opt = api.options(phi_index_offset=off, phi_index_total=total, **opt_kwargs)
    roots, caus, _, _, st = api.curves_and_caustics(star_xy, masses, kappa_s, gamma, num_phi_per_rank, tol, max_iter,
                                                    opt=opt, want_diagnostics=False)
    return roots, caus, st


def next_ranks_first_row(t):
    """t [S, n, 2] on every rank -> the first row [n, 2] of the NEXT rank (ring).  One all-gather of n x 16 bytes."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return t[0].clone()
    world, rank = dist.get_world_size(), dist.get_rank()
    mine = t[0].contiguous()
    rows = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(rows, mine)
    return rows[(rank + 1) % world]


def link_shard(api, roots):
    """Successor table of this rank's rows INCLUDING the seam: out[s][i] = column of row s+1 that continues column i
    of row s, row S being the next rank's first row.  -> (next [S, n] int32, bijective [S] int32, seam row [n, 2])."""
    import torch
    seam = next_ranks_first_row(roots)
    rows = torch.cat([roots, seam[None]], dim=0).contiguous()
    nxt, bij = api.link_rows(rows)            # cyclic by definition: the entry of the added row is not used
    return nxt[:-1].contiguous(), bij[:-1].contiguous(), seam


def crossing_map_all_ranks(api, caustics, nxt, x0, y0, pixel, nx, ny):
    """Number of caustic crossings per pixel of the WHOLE closed curve from the ranks' rows: every rank rasterises the
    segments that start in its rows (its last one ends in the next rank's first row), the integer maps are summed."""
    import torch
    import torch.distributed as dist
    seam = next_ranks_first_row(caustics)
    pts = torch.cat([caustics, seam[None]], dim=0).contiguous()
    stop = torch.full((1, nxt.shape[1]), -1, dtype=nxt.dtype, device=nxt.device)
    table = torch.cat([nxt, stop], dim=0).contiguous()
    local = api.crossing_map(pts, table, x0, y0, pixel, nx, ny, closed=False)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(local, op=dist.ReduceOp.SUM)
    return local
