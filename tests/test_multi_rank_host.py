"""World-size-2 `gloo` tests of the multi-GPU host logic on CPU.

The solve shards by phases only: rank r solves rows [r n, (r+1) n) of a grid of W n phases and there is no
data-path collective; the post-processing of the whole closed curve needs the seam (sharding.py).  What can be checked
without a GPU: the shard arithmetic tiles the grid exactly once, the max-over-ranks timing reduce, the host-only
planner on each rank's shard, and -- with `OracleBackedApi` below standing in for the binding, SAME call signatures
and (phi_index_offset, phi_index_total) contract -- that sharding.solve_shard / link_shard / crossing_map_all_ranks
under torch.distributed give the root sets, the chains and the crossing map of the single-process grid.
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


class OracleBackedApi:
    """Stands in for paper_2506_02121_b200.api in the CPU tests: the binding's function names, argument order,
    options object and return shapes (CPU tensors instead of CUDA ones), computed by the oracle.  It lets the
    multi-rank host logic run through the C-ABI call signatures without a GPU; it is test code only."""

    class _Opt:
        def __init__(self, **kw):
            self.phi_index_offset = kw.pop("phi_index_offset", 0)
            self.phi_index_total = kw.pop("phi_index_total", 0)
            self.rest = kw

    def __init__(self, oracle):
        self.o = oracle

    def options(self, **kw):
        return self._Opt(**kw)

    def curves_and_caustics(self, star_xy, masses, kappa_s, gamma, num_phi, tol=1e-12, max_iter=50, opt=None,
                            init_roots=None, out_roots=None, out_caustics=None, want_diagnostics=True, strict=True):
        off = opt.phi_index_offset if opt is not None else 0
        total = (opt.phi_index_total if opt is not None else 0) or num_phi
        xy, m = star_xy.numpy(), masses.numpy()
        rows, it, un = self.o.critical_curve_rows(xy, m, kappa_s, gamma, total, np.arange(num_phi), tol, max_iter, j_offset=off)
        caus = self.o.caustics(xy, m, kappa_s, gamma, rows)

        class St:
            unconverged_rows = int((un > 0).sum())
        return torch.from_numpy(rows), torch.from_numpy(caus), torch.from_numpy(it), torch.from_numpy(un), St()

    def link_rows(self, rows):
        nxt, bij = self.o.link_rows(rows.numpy())
        return torch.from_numpy(nxt), torch.from_numpy(bij)

    def crossing_map(self, caustics, nxt, x0, y0, pixel, nx, ny, closed=True):
        table = None if nxt is None else nxt.numpy().copy()
        if not closed:
            if table is None:
                table = np.tile(np.arange(caustics.shape[1], dtype=np.int32), (caustics.shape[0], 1))
            table[-1, :] = -1                    # the oracle closes every chain unless its table says stop
        return torch.from_numpy(self.o.crossing_map(caustics.numpy(), table, x0, y0, pixel, nx, ny))


WINDOW = (-2.2, -2.2, 4.4 / 64, 64, 64)          # crossing-map window of the cfg1 test field


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
        # the per-rank solve through the binding's call signature (offset / total contract)
        fake = OracleBackedApi(oracle)
        xy, m, R = oracle.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
        roots, caus, st = sharding.solve_shard(fake, torch.from_numpy(xy), torch.from_numpy(m), cfg.kappa_s, cfg.gamma,
                                               n_per_rank, cfg.tol, cfg.max_iter, rank, world)
        assert st.unconverged_rows == 0 and tuple(roots.shape) == (n_per_rank, 2 * cfg.N, 2)
        # the seam: my last row linked to the next rank's first row, every segment of the closed curve counted once
        nxt, bij, seam = sharding.link_shard(fake, roots)
        assert tuple(nxt.shape) == (n_per_rank, 2 * cfg.N) and bool(bij.all())
        cmap = sharding.crossing_map_all_ranks(fake, caus, nxt, *WINDOW)
        all_rows = [torch.zeros_like(roots) for _ in range(world)]
        all_next = [torch.zeros_like(nxt) for _ in range(world)]
        dist.all_gather(all_rows, roots)              # test-only gathers; the product has no such collective
        dist.all_gather(all_next, nxt)
        # timing contract: the job's time is the slowest rank's
        t = sharding.max_over_ranks(10.0 + rank)
        assert t == 10.0 + world - 1
        if rank == 0:
            np.save(os.path.join(out_dir, "rows.npy"), torch.cat(all_rows).numpy())
            np.save(os.path.join(out_dir, "next.npy"), torch.cat(all_next).numpy())
            np.save(os.path.join(out_dir, "cmap.npy"), cmap.numpy())
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_world_size_2_phase_sharding_and_seams(tmp_path, orc):
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
    # the ranks' successor tables, stacked, are the single-process table of the stacked rows (seam rows included)
    nxt_ref, bij_ref = orc.link_rows(sharded)
    assert bij_ref.all() and np.array_equal(np.load(tmp_path / "next.npy"), nxt_ref)
    # ... and the summed crossing map is the map of the whole closed curve
    caus = orc.caustics(xy, m, cfg.kappa_s, cfg.gamma, sharded)
    cmap_ref, amb = orc.crossing_map(caus, nxt_ref, *WINDOW, want_ambiguous=True)
    cmap = np.load(tmp_path / "cmap.npy")
    assert cmap_ref.max() >= 1 and np.array_equal(cmap[amb == 0], cmap_ref[amb == 0])


def test_bench_refuses_more_ranks_than_gpus():
    """python bench.py --gpus 2 on a box with fewer than 2 GPUs must fail loudly, not run one rank (or a CPU path)."""
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--num-phi", "64", "--steps", "1",
                        "--warmup", "1"], capture_output=True, text=True, env=env, timeout=300)
    if torch.cuda.is_available() and torch.cuda.device_count() >= 2:
        pytest.skip("this box has two GPUs: the launcher would start the ranks")
    assert r.returncode != 0
    assert "refusing" in (r.stderr + r.stdout) and '"metric"' not in r.stdout


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
