"""World-size-2 `gloo` test of the multi-GPU host logic on CPU.

The path shards by phases only: rank r solves rows [r n, (r+1) n) of a grid of W n phases and there is no
data-path collective.  What can be checked without a GPU: the shard arithmetic tiles the grid exactly once,
the max-over-ranks timing reduce, the host-only planner on each rank's shard, and — with the oracle standing
in for the per-rank solve — that solving each shard with (phi_index_offset, phi_index_total) and
concatenating gives the root sets of the single-process grid.
"""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

from paper_2506_02121_b200 import sharding  # noqa: E402
from paper_2506_02121_b200.configs import CONFIGS  # noqa: E402


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, n_per_rank, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        from paper_2506_02121_b200 import api
        cfg = CONFIGS["cfg1"]
        off, total = sharding.phase_shard(rank, world, n_per_rank)
        # every rank sees every shard: they tile [0, total) exactly once
        mine = torch.tensor([off, n_per_rank, total], dtype=torch.int64)
        gathered = [torch.zeros(3, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(gathered, mine)
        covered = np.zeros(total, np.int32)
        for g in gathered:
            assert int(g[2]) == total
            covered[int(g[0]):int(g[0]) + int(g[1])] += 1
        assert (covered == 1).all()
        # the host-only planner (no CUDA call) on this rank's shard
        first, centre, end = api.plan_subchains(cfg.N, n_per_rank, 0)
        assert first[0] == 0 and end[-1] == n_per_rank and (first[1:] == end[:-1]).all()
        # the per-rank solve, the oracle standing in for the GPU call with the same (offset, total) contract
        xy, m, R = oracle.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
        rows, _, un = oracle.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, total,
                                                 np.arange(n_per_rank), cfg.tol, cfg.max_iter, j_offset=off)
        assert un.sum() == 0
        mine_rows = torch.from_numpy(rows)
        all_rows = [torch.zeros_like(mine_rows) for _ in range(world)]
        dist.all_gather(all_rows, mine_rows)          # test-only gather; the product has no such collective
        # timing contract: the job's time is the slowest rank's
        t = sharding.max_over_ranks(10.0 + rank)
        assert t == 10.0 + world - 1
        if rank == 0:
            np.save(os.path.join(out_dir, "rows.npy"), torch.cat(all_rows).numpy())
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_world_size_2_phase_sharding(tmp_path, orc):
    world, n_per_rank = 2, 30
    port = _free_port()
    mp.spawn(_worker, args=(world, port, n_per_rank, str(tmp_path)), nprocs=world, join=True)
    sharded = np.load(tmp_path / "rows.npy")
    cfg = CONFIGS["cfg1"]
    xy, m, R = orc.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
    ref, _, un = orc.critical_curves(xy, m, cfg.kappa_s, cfg.gamma, world * n_per_rank, cfg.tol, cfg.max_iter)
    assert un.sum() == 0 and sharded.shape == ref.shape
    err, bij = orc.match_root_sets(sharded, ref, 1e-10)
    assert bij.all() and err.max() < 1e-12


def test_shard_arithmetic():
    assert sharding.phase_shard(0, 1, 100) == (0, 100)
    assert sharding.phase_shard(3, 8, 10000) == (30000, 80000)
    for total, world in ((10000, 8), (10, 3), (7, 7)):
        parts = sharding.split_rows(total, world)
        assert parts[0][0] == 0 and sum(n for _, n in parts) == total
        assert all(parts[i][0] + parts[i][1] == parts[i + 1][0] for i in range(world - 1))
        assert max(n for _, n in parts) - min(n for _, n in parts) <= 1
    with pytest.raises(ValueError):
        sharding.phase_shard(2, 2, 10)
    with pytest.raises(ValueError):
        sharding.split_rows(3, 4)
    assert sharding.max_over_ranks(3.5) == 3.5     # no process group: identity
