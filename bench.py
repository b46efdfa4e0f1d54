#!/usr/bin/env python
"""bench.py — converged critical-curve roots/s on the headline workload (BASELINE.json: N = 10^4 stars, fp64).

One "step" is one pass of the whole hot path over one workload, through the C-ABI:
  a0 mlcc_star_field -> a1..a7 mlcc_curves_and_caustics (caustic map fused into the Aberth kernel) -> a8 validator:
  mlcc_match_root_sets (this step's root sets against the previous step's), mlcc_vieta_residuals on every row,
  mlcc_detj_residuals on every 50th row (the full certificate of every row is run once, outside the timed region).
Every pair of the iteration is FP64 arithmetic (mlcc_options.aberth_sum_precision = 64, the library default); the
same workload with the Aberth sum in packed double-single FP32 is timed beside it (`mixed_precision`).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg4] [--num-phi M]
N > 1: one rank per GPU under torch.distributed.run (bench.py starts it itself when WORLD_SIZE is not set); the phase
grid is N times as long and rank r owns rows [r*num_phi, (r+1)*num_phi) (weak scaling, no data-path collective;
DESIGN.md "Multi-GPU").

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle on the host cores instead.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2506_02121_b200.configs import CONFIGS, HEADLINE  # noqa: E402

METRIC = "converged critical-curve roots/s"
UNIT = "roots/s"
# algorithmic flop per pair, one reciprocal counted as 1 flop
FLOP_PER_STAR_PAIR = 27.0
FLOP_PER_STAR_PAIR_NO_S1 = 25.0   # iterations without the Aberth sum do not accumulate S1 (R27)
FLOP_PER_ROOT_PAIR = 10.0
# FP64 instructions the kernels execute per pair (SASS of k_compute / k_chain; profiles/r02_k_compute_sass.md):
# star pair with the fused caustic sum 7 DADD + 7 DMUL + 10 DFMA, without S1 5 + 7 + 10; root pair 2 DADD + 4 DFMA
HW_FLOP_STAR, HW_FLOP_STAR_NO_S1, HW_FLOP_ROOT = 34.0, 32.0, 10.0
NCU_PROFILE = os.path.join(ROOT, "profiles", "r02_k_compute_ncu.csv")   # committed capture: DRAM bytes, hardware flop
DETJ_ROW_STRIDE_MAX = 64   # the timed step certifies every d-th row, d the largest divisor of the grid up to this


def detj_stride(total, off):
    """Largest d <= DETJ_ROW_STRIDE_MAX that divides the phase grid and the rank's row offset: row q of the sampled
    rows is then row q d of the grid, with phase 2 pi (q + off/d) / (total/d) exactly."""
    for d in range(min(DETJ_ROW_STRIDE_MAX, total), 0, -1):
        if total % d == 0 and off % d == 0:
            return d
    return 1


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=HEADLINE, choices=sorted(CONFIGS))
    ap.add_argument("--num-phi", type=int, default=0, help="override the number of phases (profiling runs)")
    ap.add_argument("--only-headline", action="store_true",
                    help="time the headline workload only (no other configs, no side legs, no e2e, no CPU baseline): "
                         "the form used under ncu")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config table (cfg1..cfg5)")
    ap.add_argument("--no-extras", action="store_true", help="skip mixed_precision / far_field / predicted_newton")
    ap.add_argument("--post", action="store_true",
                    help="also time the post-processing calls on the step's outputs (chain joining, closed loops, "
                         "crossing map, distance maps) and add them as `post_processing`; outside the timed region")
    ap.add_argument("--subchains", type=int, default=0)
    ap.add_argument("--order", type=int, default=-1)
    ap.add_argument("--min-lanes", type=int, default=0)
    ap.add_argument("--regime", type=int, default=0, choices=[0, 1, 2], help="mlcc_options.regime (0 auto, 1 tiled, 2 chain)")
    ap.add_argument("--aberth-sum", type=int, default=0, choices=[0, 32, 64],
                    help="arithmetic of the Aberth sum: 64 = FP64 (default), 32 = packed double-single FP32")
    ap.add_argument("--star-sums", default="direct", choices=["direct", "fmm"],
                    help="direct: O(N) star sums as BASELINE.json fixes (headline); fmm: the paper's near/far split "
                         "(PAPER.md:188-195) -- the roofline object then counts the root pairs only")
    ap.add_argument("--skip-aberth-below", type=float, default=0.0,
                    help="mlcc_options.skip_aberth_sum_below (0 = library default, negative = never skip)")
    ap.add_argument("--clock-sample-ms", type=int, default=200,
                    help="period of the NVML clock / throttle-reason samples taken during the timed region")
    ap.add_argument("--trust-predictor", action="store_true",
                    help="mlcc_options.trust_predictor = 1 in the timed steps (DESIGN.md R30; not the headline)")
    ap.add_argument("--cpu-budget-s", type=float, default=240.0,
                    help="soft bound on the CPU-baseline leg: the cfg5 sample shrinks (and says so) if the plan does not fit")
    return ap.parse_args()


class ClockSampler:
    """NVML clocks / throttle reasons sampled during the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index=0, period_ms=200):
        self.rows, self.proc, self.thread, self.gpu, self.period_ms = [], None, None, gpu_index, int(period_ms)
        self.nvml, self.handle, self.running, self.smax = None, None, False, 0.0

    def start(self):
        # In-process NVML first (four light queries per sample).  An nvidia-smi -lms loop beside the run was measured
        # to stall this process's kernel launches now and then; it is kept only as the fallback.
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nvml = pynvml
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(self.gpu)
            self.smax = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
            self.running = True
            self.proc = "nvml"
            self.thread = threading.Thread(target=self._read_nvml, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", str(self.period_ms), "-i", str(self.gpu)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read_nvml(self):
        nv, h = self.nvml, self.handle
        bits = ((nv.nvmlClocksThrottleReasonHwSlowdown, 5), (nv.nvmlClocksThrottleReasonHwThermalSlowdown, 6),
                (nv.nvmlClocksThrottleReasonSwThermalSlowdown, 7), (nv.nvmlClocksThrottleReasonSwPowerCap, 8))
        while self.running:
            try:
                row = [str(self.gpu), str(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)), str(self.smax),
                       str(nv.nvmlDeviceGetPowerUsage(h) / 1000.0), "", "", "", "", ""]
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, col in bits:
                    row[col] = "Active" if (mask & bit) else "Not Active"
                self.rows.append((time.time(), row))
            except Exception:
                pass
            time.sleep(self.period_ms / 1000.0)

    def sample_now(self):
        """One synchronous sample (used at both ends of a timed region, so that regions shorter than the sampling
        period still carry the clocks they ran at)."""
        if self.proc != "nvml":
            return
        nv, h = self.nvml, self.handle
        try:
            row = [str(self.gpu), str(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)), str(self.smax),
                   str(nv.nvmlDeviceGetPowerUsage(h) / 1000.0), "", "", "", "", ""]
            mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
            for bit, col in ((nv.nvmlClocksThrottleReasonHwSlowdown, 5), (nv.nvmlClocksThrottleReasonHwThermalSlowdown, 6),
                             (nv.nvmlClocksThrottleReasonSwThermalSlowdown, 7), (nv.nvmlClocksThrottleReasonSwPowerCap, 8)):
                row[col] = "Active" if (mask & bit) else "Not Active"
            self.rows.append((time.time(), row))
        except Exception:
            pass

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def window(self, t_begin=None, t_end=None):
        """Summary of the samples that arrived in [t_begin, t_end] (None = all of them); the sampler keeps running."""
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["clock sampler unavailable"]}
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for when, r in list(self.rows):
            if (t_begin is not None and when < t_begin) or (t_end is not None and when > t_end):
                continue
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1])); smax.append(float(r[2])); power.append(float(r[3]))
            except ValueError:
                continue
            for n, v in zip(names, r[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons),
                "source": "nvml (in-process)" if self.proc == "nvml" else "nvidia-smi -lms"}

    def stop(self):
        if not self.proc:
            return
        if self.proc == "nvml":
            self.running = False
            self.thread.join(timeout=5)
        else:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()


# ---------------------------------------------------------------------------------------------------------------
# the oracle legs (cpu_baseline, --impl reference): the only places bench.py executes oracle/
# ---------------------------------------------------------------------------------------------------------------
def oracle_cold_and_continued(cfg, num_phi, n_cont, j0=None):
    """Times the oracle as it stands: row j0 cold-started from z_i +/- 1, then n_cont rows continued from it (each
    from the row before), with their caustic points.  -> dict(seconds_cold_row, seconds_per_continued_row, ...)."""
    import oracle
    xy, m, R = oracle.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
    j0 = num_phi // 2 if j0 is None else j0
    t0 = time.perf_counter()
    r0, it0, un0 = oracle.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, num_phi, [j0], cfg.tol, cfg.max_iter)
    oracle.caustics(xy, m, cfg.kappa_s, cfg.gamma, r0)
    t_cold = time.perf_counter() - t0
    t_cont, it1 = 0.0, np.zeros(0, np.int32)
    if n_cont > 0:
        rows = [(j0 + 1 + q) % num_phi for q in range(n_cont)]
        t0 = time.perf_counter()
        r1, it1, un1 = oracle.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, num_phi, rows, cfg.tol, cfg.max_iter,
                                                  init_roots=r0[0])
        oracle.caustics(xy, m, cfg.kappa_s, cfg.gamma, r1)
        t_cont = (time.perf_counter() - t0) / n_cont
    n_r = 2 * cfg.N
    full = t_cold + (num_phi - 1) * t_cont if n_cont > 0 else None
    return {"seconds_cold_row": t_cold, "seconds_per_continued_row": t_cont if n_cont > 0 else None,
            "cold_row_iterations": int(it0[0]), "continued_row_iterations": [int(v) for v in it1[:8]],
            "rows_timed": 1 + n_cont, "seconds": t_cold + n_cont * t_cont,
            "extrapolated_full_set_s": full, "extrapolated": True,
            "roots_per_s": (num_phi * n_r / full) if full else n_r / t_cold,
            "cores": oracle.num_threads(),
            "sample": f"row {j0} of {num_phi} cold-started from z_i+/-1, then {n_cont} rows continued from it, with their "
                      f"caustic points; full set = cold row + ({num_phi} - 1) x continued row (linear extrapolation)"}


def oracle_full(cfg, num_phi):
    """The oracle on the whole grid (row 0 cold, every other row continued), with the caustic points."""
    import oracle
    xy, m, R = oracle.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
    t0 = time.perf_counter()
    roots, iters, unconv = oracle.critical_curves(xy, m, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter)
    oracle.caustics(xy, m, cfg.kappa_s, cfg.gamma, roots)
    dt = time.perf_counter() - t0
    return {"seconds_full_set": dt, "extrapolated": False, "roots_per_s": num_phi * 2 * cfg.N / dt,
            "cores": oracle.num_threads(), "rows_timed": num_phi,
            "iterations_cold_row": int(iters[0]), "iterations_per_continued_row_mean": float(iters[1:].mean()) if num_phi > 1 else None,
            "sample": f"all {num_phi} rows (row 0 cold-started, the others continued) with their caustic points"}


def run_reference(args, cfg, num_phi):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the workload per step."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    # per step: one cold row + n_cont continued rows (about 5 s at N = 10^4 on 16 cores)
    n_cont = 8 if cfg.N >= 1000 else min(num_phi - 1, 199)
    for _ in range(args.warmup):
        oracle_cold_and_continued(cfg, num_phi, 0 if cfg.N >= 5000 else n_cont)
    t_all, t_cold, t_cont, cores, sample = 0.0, 0.0, 0.0, 1, ""
    for _ in range(args.steps):
        r = oracle_cold_and_continued(cfg, num_phi, n_cont)
        t_all += r["seconds"]
        t_cold += r["seconds_cold_row"]
        t_cont += r["seconds_per_continued_row"] or 0.0
        cores, sample = r["cores"], r["sample"]
    t_cold /= args.steps
    t_cont /= args.steps
    n_r = 2 * cfg.N
    full = t_cold + (num_phi - 1) * t_cont
    value = num_phi * n_r / full
    cpu = {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
           "seconds_per_cold_row": t_cold, "seconds_per_continued_row": t_cont, "extrapolated_full_set_s": full,
           "extrapolated": True, "sampled_roots_per_s": (1 + n_cont) * n_r * args.steps / t_all}
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_all / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg.name}: N={cfg.N}, num_phi={num_phi} (bounded sample per step, value extrapolated "
                                   f"to the full set)", "sample": sample, "extrapolated": True},
            "cpu_baseline": cpu,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------------------------
# --gpus N: start the ranks ourselves when nobody did
# ---------------------------------------------------------------------------------------------------------------
def relaunch_under_torchrun(args):
    """python bench.py --gpus N (N > 1) without WORLD_SIZE: run the same command under torch.distributed.run with one
    rank per GPU.  Fails loudly when the box has fewer GPUs: N ranks never share fewer devices."""
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit(f"bench.py --gpus {args.gpus}: this box has {have} CUDA device(s); refusing to run "
                         f"{args.gpus} ranks on fewer GPUs")
    port = 29500 + (os.getpid() % 2000)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


# ---------------------------------------------------------------------------------------------------------------
# the GPU legs
# ---------------------------------------------------------------------------------------------------------------
class Workbench:
    """Device buffers and the timed step of one workload."""

    def __init__(self, api, torch, cfg, num_phi, opt, phi_off, phi_total):
        self.api, self.torch, self.cfg, self.num_phi, self.opt = api, torch, cfg, num_phi, opt
        self.phi_off, self.phi_total = phi_off, phi_total
        self.n_r = 2 * cfg.N
        self.roots = torch.empty((num_phi, self.n_r, 2), dtype=torch.float64, device="cuda")
        self.prev = torch.empty_like(self.roots)
        self.caus = torch.empty_like(self.roots)
        self.last = {}
        self.stride = detj_stride(phi_total if phi_total > 0 else num_phi, phi_off)
        self.sample_rows = torch.arange(0, num_phi, self.stride, device="cuda")

    def step(self):
        api, cfg = self.api, self.cfg
        xy, m, R = api.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
        _, _, _, _, st = api.curves_and_caustics(xy, m, cfg.kappa_s, cfg.gamma, self.num_phi, cfg.tol, cfg.max_iter,
                                                 opt=self.opt, out_roots=self.roots, out_caustics=self.caus,
                                                 want_diagnostics=False)
        # the very first call has no previous step to compare with: it checks the sets against themselves
        err, bij = api.match_root_sets(self.roots, self.prev if self.last else self.roots, 1e-10)
        v1, v2 = api.vieta_residuals(xy, m, cfg.kappa_s, cfg.gamma, self.roots, self.phi_off, self.phi_total)
        # det J / Newton-residual certificate on every stride-th row: the rows are gathered and certified by ONE call on
        # the coarser grid (offset / stride, total / stride), which has exactly their phases
        total = self.phi_total if self.phi_total > 0 else self.num_phi
        rn, rd, _ = api.detj_residuals(xy, m, cfg.kappa_s, cfg.gamma, self.roots[self.sample_rows],
                                       self.phi_off // self.stride, total // self.stride)
        self.last.update(stats=st, err=err, bij=bij, v1=v1, v2=v2, rn=rn, rd=rd, xy=xy, m=m)
        return st

    def check(self):
        last, st = self.last, self.last["stats"]
        assert bool(last["bij"].all()), "validator: this step's root sets differ from the previous step's"
        assert float(last["v1"].max()) < 1e-12 and float(last["v2"].max()) < 1e-12, "validator: a row fails Vieta's sums"
        assert float(last["rd"].max()) <= 1.0, "validator: det J above the scale-aware bound on a sampled row"
        assert float(last["rn"].max()) < 1e-11, "validator: Newton residual of a sampled root above 1e-11"
        assert st.unconverged_rows == 0 and st.degenerate_roots == 0

    def certificate_all_rows(self):
        """mlcc_detj_residuals on EVERY row of the last step's outputs (outside the timed region)."""
        torch, api, cfg = self.torch, self.api, self.cfg
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        rn, rd, _ = api.detj_residuals(self.last["xy"], self.last["m"], cfg.kappa_s, cfg.gamma, self.roots,
                                       self.phi_off, self.phi_total)
        e1.record()
        torch.cuda.synchronize()
        return {"rows": self.num_phi, "max_newton_residual": float(rn.max()), "max_detj_over_bound": float(rd.max()),
                "rows_certified": int((rd <= 1.0).sum()), "ms": e0.elapsed_time(e1),
                "bound": "|1/mu| <= 1e-10 + 4 (1-kappa_s) |F'| 2^-52 (1+|z|) (SURVEY.md 0.2)"}


def flop_model(cfg, st, star_sums, mode):
    """Algorithmic and hardware-instruction flop of one call's counters, split by the pipe that executes them."""
    n_r = 2 * cfg.N
    with_A = st.root_pairs / float(n_r - 1)
    without_A = st.root_iterations - with_A
    star_alg = 0.0 if star_sums == "fmm" else FLOP_PER_STAR_PAIR * cfg.N * with_A + FLOP_PER_STAR_PAIR_NO_S1 * cfg.N * without_A
    star_hw = 0.0 if star_sums == "fmm" else HW_FLOP_STAR * cfg.N * with_A + HW_FLOP_STAR_NO_S1 * cfg.N * without_A
    root_alg = FLOP_PER_ROOT_PAIR * st.root_pairs
    survey = (FLOP_PER_STAR_PAIR * cfg.N + FLOP_PER_ROOT_PAIR * (n_r - 1)) * st.root_iterations
    if mode == 32:
        return {"fp64": star_alg, "fp32": root_alg, "hw_fp64": star_hw, "survey": survey}
    return {"fp64": star_alg + root_alg, "fp32": 0.0, "hw_fp64": star_hw + HW_FLOP_ROOT * st.root_pairs, "survey": survey}


def time_workload(api, torch, dist, world, sampler, cfg, num_phi, opt, phi_off, phi_total, steps, warmup, star_sums):
    """W warm-up steps, K timed steps bracketed by barrier + synchronize; -> (Workbench, dict of measurements)."""
    wb = Workbench(api, torch, cfg, num_phi, opt, phi_off, phi_total)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(warmup, 1)):
        wb.step()
        wb.prev.copy_(wb.roots)
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    acc = {"solve_ms": 0.0, "launches": 0, "fp64": 0.0, "fp32": 0.0, "hw_fp64": 0.0, "survey": 0.0, "iterations": 0}
    barrier()
    t_begin = time.time()
    ev0.record()
    for i_step in range(steps):
        if sampler is not None and i_step == steps - 1:
            sampler.sample_now()          # launches of the earlier steps are still running: a sample under load
        st = wb.step()
        f = flop_model(cfg, st, star_sums, st.aberth_sum_precision)
        acc["solve_ms"] += st.solve_ms
        acc["launches"] += st.kernel_launches + 3 + 1 + 2 + 1   # star field (3), matcher, Vieta sums (2), det J
        acc["iterations"] += st.total_iterations
        for k in ("fp64", "fp32", "hw_fp64", "survey"):
            acc[k] += f[k]
    ev1.record()
    if sampler is not None:
        sampler.sample_now()              # the device is still working through the last step's launches
    barrier()
    t_end = time.time()
    ms = ev0.elapsed_time(ev1)
    wb.check()
    t = torch.tensor([ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    acc["ms_per_step"] = float(t.item()) / steps
    acc["clocks"] = sampler.window(t_begin, t_end) if sampler is not None else None
    acc["steps"], acc["warmup"] = steps, max(warmup, 1)
    return wb, acc


def roofline_of(acc, peak64, peak32, mode, survey_ok=True):
    s = acc["solve_ms"] * 1e-3
    if s <= 0:
        return {}
    f64 = acc["fp64"] / s / 1e12
    f32 = acc["fp32"] / s / 1e12
    return {"fp64_algorithmic_tflops": f64, "fp64_frac": f64 / peak64 if peak64 else None,
            "fp32_algorithmic_tflops": f32, "fp32_frac": (f32 / peak32 if peak32 else None) if mode == 32 else 0.0,
            "combined_frac": ((f64 / peak64 if peak64 else 0.0) + (f32 / peak32 if (peak32 and mode == 32) else 0.0)),
            "hw_fp64_frac_model": acc["hw_fp64"] / s / 1e12 / peak64 if peak64 else None,
            "frac_with_survey_accounting": acc["survey"] / s / 1e12 / peak64 if (peak64 and mode != 32 and survey_ok) else None}


def ncu_capture_summary():
    """DRAM bytes and hardware FP64 flop of the dominant kernel from the committed ncu capture (if present)."""
    if not os.path.exists(NCU_PROFILE):
        return None
    import csv
    rows = list(csv.DictReader(open(NCU_PROFILE)))
    full = [r for r in rows if r.get("kind") == "full_iteration"]
    if not full:
        return None
    r = full[0]
    return {"source": os.path.relpath(NCU_PROFILE, ROOT), "kernel": r["kernel"], "launch_ms": float(r["duration_ms"]),
            "dram_bytes": float(r["dram_bytes_read"]) + float(r["dram_bytes_write"]),
            "hw_fp64_frac": float(r["hw_fp64_frac"]), "fp64_pipe_pct": float(r["fp64_pipe_pct"]),
            "issue_active_pct": float(r["issue_active_pct"])}


def iteration_histograms(api, torch, cfg, num_phi, opt_kwargs, phi_off, phi_total):
    """SURVEY.md §5 "Metrics": iterations per row for cold and continued rows (PAPER.md:180-182 quotes 30-50 and 20-30
    for the paper's tolerance and seeds), and the unfrozen roots entering each iteration of a cold row."""
    xy, m, R = api.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
    opt = api.options(**opt_kwargs)
    _, iters, unconv, st = api.critical_curves_ex(xy, m, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter, opt=opt)
    iters = iters.cpu().numpy()
    first, centre, end = api.plan_subchains(cfg.N, num_phi, st.subchains)
    cold = np.zeros(num_phi, bool)
    cold[centre] = True

    def hist(v):
        u, c = np.unique(v, return_counts=True)
        return {str(int(a)): int(b) for a, b in zip(u, c)}

    out = {"cold_rows": hist(iters[cold]), "continued_rows": hist(iters[~cold]),
           "paper": "30-50 cold, 20-30 continued (PAPER.md:180-182: tol 1e-9 theta_star or |mu| > 1e9, previous row as seed)"}
    # unfrozen roots after i iterations of one cold row = out_unconverged of a 1-row call capped at max_iter = i
    j0 = int(centre[0])
    total = phi_total if phi_total > 0 else num_phi
    active = [2 * cfg.N]
    for i in range(1, cfg.max_iter + 1):
        kw = dict(opt_kwargs)
        kw.update(phi_index_offset=phi_off + j0, phi_index_total=total, num_subchains=1)
        _, _, un, _ = api.critical_curves_ex(xy, m, cfg.kappa_s, cfg.gamma, 1, cfg.tol, i, opt=api.options(**kw), strict=False)
        active.append(int(un[0]))
        if active[-1] == 0:
            break
    out["active_roots_by_iteration_cold_row"] = active
    return out


def main():
    args = parse()
    cfg = CONFIGS[args.workload]
    num_phi = args.num_phi or cfg.num_phi
    if args.impl == "reference":
        run_reference(args, cfg, num_phi)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        relaunch_under_torchrun(args)

    import torch
    import torch.distributed as dist
    from paper_2506_02121_b200 import api

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    if world != args.gpus:
        raise SystemExit(f"bench.py --gpus {args.gpus} but WORLD_SIZE={world}: start one rank per GPU")
    if torch.cuda.device_count() < int(os.environ.get("LOCAL_WORLD_SIZE", world)):
        raise SystemExit(f"{world} ranks but only {torch.cuda.device_count()} CUDA device(s): ranks never share a GPU")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    api.lib()
    if args.only_headline:
        args.no_e2e = args.no_cpu_baseline = args.no_configs = args.no_extras = True
    n_r = 2 * cfg.N
    from paper_2506_02121_b200 import sharding
    phi_off, phi_total = sharding.phase_shard(rank, world, num_phi)
    base_kw = dict(num_subchains=args.subchains, predictor_order=args.order, min_lanes_per_root=args.min_lanes,
                   skip_aberth_sum_below=args.skip_aberth_below, regime=args.regime)
    head_kw = dict(base_kw, phi_index_offset=phi_off, phi_index_total=phi_total, aberth_sum_precision=args.aberth_sum,
                   star_sum_mode=api.MLCC_STAR_SUMS_FMM if args.star_sums == "fmm" else api.MLCC_STAR_SUMS_DIRECT,
                   trust_predictor=1 if args.trust_predictor else 0)
    opt = api.options(**head_kw)

    # The clock sampler is started BEFORE the warm-up (attaching to the driver can stall launches for a moment); only the
    # samples inside each timed region are reported.
    sampler = ClockSampler(local_rank, args.clock_sample_ms) if (rank == 0 and args.clock_sample_ms > 0) else None
    if sampler:
        sampler.start()

    # ---- headline: K timed steps of the workload ----
    wb, acc = time_workload(api, torch, dist, world, sampler, cfg, num_phi, opt, phi_off, phi_total, args.steps,
                            args.warmup, args.star_sums)
    st = wb.last["stats"]
    mode = st.aberth_sum_precision
    ms_per_step = acc["ms_per_step"]
    value = world * num_phi * n_r / (ms_per_step * 1e-3)

    # ---- roofline of the dominant kernel (the Aberth iteration): FP64 ALU bound; denominators measured here ----
    peak64 = api.fp64_peak(50.0) if rank == 0 else 0.0
    peak32 = api.fp64_issue_probe(4, 20.0) if rank == 0 else 0.0
    props = torch.cuda.get_device_properties(local_rank)
    sm_count = props.multi_processor_count
    sm_max_mhz = (acc["clocks"] or {}).get("sm_max_mhz") or 1965.0
    nominal64 = sm_count * 64 * 2 * sm_max_mhz * 1e6 / 1e12     # SMs x FP64 lanes x 2 flop x max SM clock
    rf = roofline_of(acc, peak64, peak32, mode, survey_ok=(args.star_sums == "direct" and not args.trust_predictor))
    ncu = ncu_capture_summary() if (args.workload == "cfg4" and args.star_sums == "direct") else None
    kernel = "mlcc::k_chain (chain regime)" if st.regime == api.MLCC_REGIME_CHAIN else "mlcc::k_compute (Aberth iteration, tiled regime)"
    roofline = {"bound": "alu", "kernel": kernel,
                "achieved": rf.get("fp64_algorithmic_tflops"), "peak": peak64, "unit": "TFLOP/s",
                "frac": rf.get("fp64_frac"),
                "fp64_frac": rf.get("fp64_frac"), "fp32_frac": rf.get("fp32_frac"), "combined_frac": rf.get("combined_frac"),
                "fp32_peak": peak32, "hw_fp64_frac_model": rf.get("hw_fp64_frac_model"),
                "frac_with_survey_accounting": rf.get("frac_with_survey_accounting"),
                "frac_of_nominal": (rf.get("fp64_algorithmic_tflops") / nominal64) if rf.get("fp64_algorithmic_tflops") else None,
                "peak_source": "measured on this GPU in this run: mlcc_fp64_peak (dependent-free 2-source DFMA loop) and "
                               f"mlcc_fp64_issue_probe form 4 (packed FP32 FMAs); nominal FP64 {nominal64:.1f} TFLOP/s = "
                               f"{sm_count} SMs x 64 lanes x 2 x {sm_max_mhz / 1e3:.3f} GHz (SM count from the device)",
                "algorithmic_flop_per_launch": acc["fp64"] / max(acc["iterations"], 1),
                "avg_launch_ms": acc["solve_ms"] / max(acc["iterations"], 1),
                "note": "achieved = algorithmic flop executed in FP64 (27 per star pair, 25 where S1 is not needed, 10 per "
                        "root pair EVALUATED when the Aberth sum is FP64; a reciprocal counts 1) / device time of the whole "
                        "solve (every launch of the call), CUDA events on the launch stream. fp32_frac = root-pair flop "
                        "executed in packed FP32 / the measured packed-FP32 peak (0 with the FP64 Aberth sum); combined_frac "
                        "= sum of work_i / peak_i over the solve time. hw_fp64_frac_model counts the DADD + DMUL + 2 DFMA the "
                        "kernels execute per pair (34 / 32 / 10) instead of the algorithmic 27 / 25 / 10; the ncu counters "
                        "of a full-iteration launch are in `ncu`",
                "traffic": ncu["dram_bytes"] if ncu else None,
                "traffic_source": ncu["source"] if ncu else None,
                "ncu": ncu}
    if rank == 0 and not args.only_headline:
        probes = {name: api.fp64_issue_probe(form, 20.0) for form, name in
                  ((1, "dfma_3_distinct_sources"), (2, "dadd_2_sources"), (3, "dfma_2_sources_interleaved_with_ffma2"))}
        roofline["issue_model"] = {"unit": "2 x FP64 instructions/s / 1e12", "dfma_2_sources (= peak)": peak64, **probes}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None,
            "dtype": "f64" if mode == 64 else "f64 (star sums, update) + packed double-single f32 (Aberth sum over roots)",
            "data": "synthetic",
            "config": {"workload": f"{cfg.name}: N={cfg.N} stars, {num_phi} phases per GPU, kappa_star={cfg.kappa_star}, "
                                   f"kappa_s={cfg.kappa_s}, gamma={cfg.gamma}, tol={cfg.tol}, max_iter={cfg.max_iter}, seed={cfg.seed}",
                       "step": "star_field + curves_and_caustics (fused) + match_root_sets + vieta_residuals + "
                               f"detj_residuals on every {wb.stride}th row",
                       "aberth_sum_precision": mode, "star_sums": args.star_sums, "trust_predictor": bool(args.trust_predictor),
                       "regime": "chain" if st.regime == api.MLCC_REGIME_CHAIN else "tiled",
                       "subchains": st.subchains, "predictor_order": st.predictor_order,
                       "l2": f"inputs larger than L2: each step writes {2 * num_phi * n_r * 16 / 1e9:.2f} GB of roots and caustics "
                             f"and reads a {num_phi * n_r * 16 / 1e9:.2f} GB comparison set (L2 is 126 MB)",
                       "seconds_per_curve_set": st.solve_ms * 1e-3,
                       "aberth_iterations_per_step": st.total_iterations,
                       "root_iterations_per_root": st.root_iterations / float(num_phi * n_r)},
            "gpu_launches": int(acc["launches"]), "clocks": acc["clocks"], "roofline": roofline}

    single = world == 1 and rank == 0
    # ---- full certificate of the headline outputs (every row), outside the timed region ----
    if single and not args.only_headline:
        line["certificate"] = wb.certificate_all_rows()

    # ---- end to end through the host-buffer C-ABI call (pinned host memory both ways) ----
    if not args.no_e2e:
        gxy, gm, _ = api.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
        p_xy = gxy.cpu().pin_memory()     # the user's host arrays (allocated outside the timed region)
        p_m = gm.cpu().pin_memory()
        h_roots = torch.empty((num_phi, n_r, 2), dtype=torch.float64, pin_memory=True)
        h_caus = torch.empty((num_phi, n_r, 2), dtype=torch.float64, pin_memory=True)
        api.curves_and_caustics_host(p_xy, p_m, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter, opt=opt,
                                     out_roots=h_roots, out_caustics=h_caus)       # warm-up
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        n_e2e = max(1, min(args.steps, 2))
        for _ in range(n_e2e):
            api.curves_and_caustics_host(p_xy, p_m, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter, opt=opt,
                                         out_roots=h_roots, out_caustics=h_caus)
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) / n_e2e
        te = torch.tensor([dt], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        same = bool(torch.equal(h_roots, wb.roots.cpu())) if single else None
        line["e2e"] = {"value": world * num_phi * n_r / float(te.item()), "unit": UNIT,
                       "h2d_bytes_per_step": int(p_xy.numel() * 8 + p_m.numel() * 8),
                       "d2h_bytes_per_step": int(h_roots.numel() * 8 + h_caus.numel() * 8),
                       "seconds_per_step": float(te.item()), "same_bits_as_device_path": same,
                       "call": "mlcc_curves_and_caustics_host (host pointers; device allocation + H2D + solve + caustics + "
                               "D2H inside the timed call; the pinned host arrays themselves are allocated before it)"}
        del h_roots, h_caus
    else:
        line["e2e"] = None

    # ---- the same workload with other arithmetic / algorithms, outside the headline's timed region ----
    if single and not args.no_extras and args.star_sums == "direct" and not args.trust_predictor:
        def side(label_kw, steps=1, warmup=1, star_sums="direct"):
            kw = dict(head_kw)
            kw.update(label_kw)
            wb2, acc2 = time_workload(api, torch, dist, 1, sampler, cfg, num_phi, api.options(**kw), phi_off, phi_total,
                                      steps, warmup, star_sums)
            st2 = wb2.last["stats"]
            err2, bij2 = api.match_root_sets(wb2.roots, wb.roots, 1e-10)
            out = {"value": num_phi * n_r / (acc2["ms_per_step"] * 1e-3), "unit": UNIT, "ms_per_step": acc2["ms_per_step"],
                   "seconds_per_curve_set": st2.solve_ms * 1e-3,
                   "matches_headline_root_sets": bool(bij2.all()), "max_abs_dz_vs_headline": float(err2.max()),
                   "root_iterations_per_root": st2.root_iterations / float(num_phi * n_r),
                   "root_iterations_with_aberth_sum_per_root": st2.root_pairs / float(n_r - 1) / float(num_phi * n_r),
                   "unconverged_rows": st2.unconverged_rows, "clocks": acc2["clocks"]}
            out.update(roofline_of(acc2, peak64, peak32, st2.aberth_sum_precision,
                                   survey_ok=(star_sums == "direct" and not kw.get("trust_predictor"))))
            del wb2
            torch.cuda.empty_cache()
            return out

        other = 32 if mode == 64 else 64
        line["mixed_precision" if other == 32 else "headline_fp64"] = dict(
            side({"aberth_sum_precision": other, "regime": api.MLCC_REGIME_TILED if other == 32 else args.regime}),
            note=("the same step with the Aberth sum over roots in packed double-single FP32 (mlcc_options."
                  "aberth_sum_precision = 32): A only steers the convergence rate, the fixed point F = 0 and the freeze "
                  "test do not see it (DESIGN.md R19); its root-pair flop are divided by the packed-FP32 peak")
            if other == 32 else "the same step with every pair in FP64")
        line["far_field"] = dict(side({"star_sum_mode": api.MLCC_STAR_SUMS_FMM}, star_sums="fmm"),
                                 note="star_sum_mode = MLCC_STAR_SUMS_FMM (PAPER.md:188-195): stars of the 5x5 nodes around a "
                                      "root directly, the rest from the node's order-31 Taylor series; the Aberth sum stays "
                                      "direct. Not the headline: BASELINE.json fixes direct O(N) star sums")
        line["predicted_newton"] = {
            "note": "trust_predictor = 1 (DESIGN.md R30): rows seeded by the cubic predictor start with Newton steps; a step "
                    "above 1e-8 is discarded and that root gets the full Aberth iteration. Not the headline",
            "direct_star_sums": side({"trust_predictor": 1}),
            "far_field_star_sums": side({"trust_predictor": 1, "star_sum_mode": api.MLCC_STAR_SUMS_FMM}, star_sums="fmm")}

    # ---- iteration histograms of the headline workload (one diagnostics run, outside the timed region) ----
    if single and not args.only_headline:
        line["iterations"] = iteration_histograms(api, torch, cfg, num_phi, head_kw, phi_off, phi_total)

    # ---- post-processing of the timed step's outputs, outside the timed region ----
    if args.post and single:
        roots, caus = wb.roots, wb.caus

        def timed(f, reps=3):
            f()
            best, out = None, None
            for _ in range(reps):
                torch.cuda.synchronize()
                p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                p0.record()
                out = f()
                p1.record()
                torch.cuda.synchronize()
                t_ms = p0.elapsed_time(p1)
                best = t_ms if best is None or t_ms < best else best
            return best, out

        n_pix = 2048
        half = 0.134 * (cfg.N / cfg.kappa_star) ** 0.5          # 60 theta_star wide at cfg4
        pixel = 2 * half / n_pix
        t_link, (nxt, lbij) = timed(lambda: api.link_rows(roots))
        t_loops, (col, end, lid, cnt) = timed(lambda: api.closed_loops(nxt))
        t_order, ordered = timed(lambda: api.order_by_chain(roots, col))
        del ordered
        t_cross, cmap = timed(lambda: api.crossing_map(caus, nxt, -half, -half, pixel, n_pix, n_pix))
        t_edt, dmap = timed(lambda: api.distance_map(cmap, pixel))
        t_dir, ddir = timed(lambda: api.directional_distance_map(cmap, pixel, 0, 1))
        gather_bytes = roots.numel() * 8 * 2 + col.numel() * 4
        line["post_processing"] = {
            "unit": "ms per call (best of 3, CUDA events)", "rows": num_phi, "roots_per_row": n_r,
            "map": f"{n_pix} x {n_pix} pixels of {pixel:.4f} theta_star",
            "link_rows": t_link, "rows_not_bijective": int((lbij == 0).sum()),
            "closed_loops": t_loops, "num_loops": int(cnt.item()), "chains_not_closed": int((lid < 0).sum()),
            "order_by_chain": t_order, "order_by_chain_GBps": gather_bytes / t_order / 1e6,
            "crossing_map": t_cross, "max_crossings": int(cmap.max()),
            "distance_map": t_edt, "directional_distance_map_(0,1)": t_dir,
            "rays_that_met_a_caustic": float((ddir > 0).double().mean())}
        del nxt, col, cmap, dmap, ddir

    # ---- all five configs, each as its own timed step sequence (BASELINE.json: "all five configs") ----
    head_summary = {"seconds_per_curve_set": st.solve_ms * 1e-3, "roots_per_s": value, "ms_per_step": ms_per_step,
                    "roofline_frac": rf.get("fp64_frac"), "hw_fp64_frac_model": rf.get("hw_fp64_frac_model"),
                    "root_iterations_per_root": st.root_iterations / float(num_phi * n_r),
                    "unconverged_rows": st.unconverged_rows, "vieta_max": max(float(wb.last["v1"].max()), float(wb.last["v2"].max())),
                    "detj_max_over_bound": (line.get("certificate") or {}).get("max_detj_over_bound"),
                    "newton_residual_max": (line.get("certificate") or {}).get("max_newton_residual"),
                    "regime": "chain" if st.regime == api.MLCC_REGIME_CHAIN else "tiled", "subchains": st.subchains,
                    "steps": args.steps, "warmup": args.warmup, "clocks": acc["clocks"]}
    del wb
    torch.cuda.empty_cache()
    if single and not args.no_configs:
        table = {}
        for name in sorted(CONFIGS):
            c = CONFIGS[name]
            if name == args.workload and num_phi == c.num_phi:
                table[name] = head_summary
                continue
            k_steps, k_warm = (1, 1) if c.N >= 20000 else (3, 2)
            wbc, accc = time_workload(api, torch, dist, 1, sampler, c, c.num_phi, api.options(**base_kw), 0, 0, k_steps,
                                      k_warm, "direct")
            stc = wbc.last["stats"]
            rfc = roofline_of(accc, peak64, peak32, stc.aberth_sum_precision)
            cert = wbc.certificate_all_rows()
            table[name] = {"seconds_per_curve_set": accc["solve_ms"] * 1e-3 / k_steps,
                           "roots_per_s": c.num_phi * 2 * c.N / (accc["ms_per_step"] * 1e-3),
                           "ms_per_step": accc["ms_per_step"], "roofline_frac": rfc.get("fp64_frac"),
                           "hw_fp64_frac_model": rfc.get("hw_fp64_frac_model"),
                           "root_iterations_per_root": stc.root_iterations / float(c.num_phi * 2 * c.N),
                           "unconverged_rows": stc.unconverged_rows,
                           "vieta_max": max(float(wbc.last["v1"].max()), float(wbc.last["v2"].max())),
                           "detj_max_over_bound": cert["max_detj_over_bound"], "newton_residual_max": cert["max_newton_residual"],
                           "certificate_ms": cert["ms"],
                           "regime": "chain" if stc.regime == api.MLCC_REGIME_CHAIN else "tiled", "subchains": stc.subchains,
                           "steps": k_steps, "warmup": k_warm, "clocks": accc["clocks"]}
            del wbc
            torch.cuda.empty_cache()
        line["configs"] = table

    if sampler:
        sampler.stop()

    # ---- CPU baseline: the oracle as it stands on the host cores (rank 0, N = 1 only), BASELINE.md §3 ----
    if single and not args.no_cpu_baseline:
        t_leg = time.perf_counter()
        per = {}
        for name in sorted(CONFIGS):
            c = CONFIGS[name]
            if c.N <= 2000:
                per[name] = oracle_full(c, c.num_phi)
            else:
                n_cont = 8
                if c.N >= 20000:
                    # planned: cold row + 8 continued rows; shrink (and say so) if the budget does not allow it.  A
                    # continued row costs about (N / 10^4)^2 times cfg4's.
                    ref = per.get("cfg4")
                    if ref and ref.get("seconds_per_continued_row"):
                        scale = (c.N / 1e4) ** 2
                        est = ref["seconds_cold_row"] * scale + 8 * ref["seconds_per_continued_row"] * scale
                        left = args.cpu_budget_s - (time.perf_counter() - t_leg)
                        while n_cont > 2 and est > left:
                            n_cont -= 1
                            est -= ref["seconds_per_continued_row"] * scale
                per[name] = oracle_cold_and_continued(c, c.num_phi, n_cont)
                per[name]["continued_rows_planned"] = 8
        h = per[args.workload] if (args.workload in per and num_phi == cfg.num_phi) else oracle_cold_and_continued(cfg, num_phi, 8)
        line["cpu_baseline"] = {"value": h["roots_per_s"], "unit": UNIT, "cores": h["cores"], "kind": "oracle",
                                "sample": h["sample"], "extrapolated": h["extrapolated"],
                                "seconds_per_cold_row": h.get("seconds_cold_row"),
                                "seconds_per_continued_row": h.get("seconds_per_continued_row"),
                                "extrapolated_full_set_s": h.get("extrapolated_full_set_s", h.get("seconds_full_set")),
                                "build": "gcc -O3 -march=native -ffp-contract=off -fopenmp (oracle/build.py)",
                                "configs": per, "leg_seconds": time.perf_counter() - t_leg}
    else:
        line.setdefault("cpu_baseline", None)

    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
