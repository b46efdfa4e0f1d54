#!/usr/bin/env python
"""bench.py — converged critical-curve roots/s on the headline workload (BASELINE.json: N = 10^4 stars, fp64).

One "step" is one pass of the whole hot path over the cfg4 workload, through the C-ABI:
  a0 mlcc_star_field -> a1..a7 mlcc_curves_and_caustics (caustic map fused into the Aberth kernel) -> a8 mlcc_match_root_sets
(the validator compares the step's root sets with those of the previous step: the run-to-run check).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg4] [--num-phi M]
N > 1: launched by torch.distributed.run, one rank per GPU; the phase grid is N times as long and rank r owns
rows [r*num_phi, (r+1)*num_phi) (weak scaling, no data-path collective).

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
FLOP_PER_STAR_PAIR = 27.0   # algorithmic flop per (root, star) pair, 1 reciprocal = 1 flop
FLOP_PER_ROOT_PAIR = 10.0   # per (root, root) pair
NCU_DRAM_BYTES_FULL_ITERATION = 11_930_880 + 6_912     # profiles/r01_k_compute_ncu.md C (launch 4: read + write)
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # SMs x FP64 lanes x 2 flop x max SM clock


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=HEADLINE, choices=sorted(CONFIGS))
    ap.add_argument("--num-phi", type=int, default=0, help="override the number of phases (profiling runs)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--post", action="store_true",
                    help="also time the post-processing calls on the step's outputs (chain joining, closed loops, "
                         "crossing map, distance maps) and add them as `post_processing`; outside the timed region")
    ap.add_argument("--subchains", type=int, default=0)
    ap.add_argument("--order", type=int, default=-1)
    ap.add_argument("--min-lanes", type=int, default=0)
    ap.add_argument("--aberth-sum", type=int, default=0, choices=[0, 32, 64],
                    help="arithmetic of the Aberth sum: 32 = double-single FP32 (default), 64 = FP64 seed form")
    ap.add_argument("--star-sums", default="direct", choices=["direct", "fmm"],
                    help="direct: O(N) star sums as BASELINE.json fixes (headline); fmm: the paper's near/far split "
                         "(PAPER.md:188-195) -- the roofline object then counts the root pairs only")
    ap.add_argument("--skip-aberth-below", type=float, default=0.0,
                    help="mlcc_options.skip_aberth_sum_below (0 = library default, negative = never skip)")
    ap.add_argument("--clock-sample-ms", type=int, default=200,
                    help="period of the nvidia-smi clock / throttle-reason samples taken during the timed region")
    ap.add_argument("--trust-predictor", action="store_true",
                    help="mlcc_options.trust_predictor = 1 in the timed steps (DESIGN.md R30; not the headline)")
    ap.add_argument("--separate-caustics", action="store_true",
                    help="run mlcc_critical_curves_ex + mlcc_caustics instead of the fused call")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index=0, period_ms=200):
        self.rows, self.proc, self.thread, self.gpu, self.period_ms = [], None, None, gpu_index, int(period_ms)
        self.nvml, self.handle, self.running, self.smax = None, None, False, 0.0

    def start(self):
        # In-process NVML first (four light queries per sample).  An nvidia-smi -lms loop beside the run was measured
        # to stall this process's kernel launches now and then (profiles/r01_bench_cfg4.md: 85 ms of non-solve time per
        # step without it, 85-260 ms with it); it is kept only as the fallback when pynvml is not importable.
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

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self, t_begin=None, t_end=None):
        """Summary of the samples that arrived in [t_begin, t_end] (the timed region; None = all of them)."""
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        if self.proc == "nvml":
            self.running = False
            self.thread.join(timeout=5)
        else:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for when, r in self.rows:
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


def oracle_sample(cfg, rows, num_phi_total, j_offset=0):
    """Times the oracle as it stands on `rows` (first row cold-started, the rest continued). -> (seconds, roots)."""
    import oracle
    xy, m, R = oracle.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
    t0 = time.perf_counter()
    roots, iters, unconv = oracle.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, num_phi_total, rows, cfg.tol,
                                                      cfg.max_iter, j_offset=j_offset)
    oracle.caustics(xy, m, cfg.kappa_s, cfg.gamma, roots)
    dt = time.perf_counter() - t0
    return dt, len(rows) * 2 * cfg.N, oracle.num_threads()


def run_reference(args, cfg, num_phi):
    """--impl reference: the CPU oracle on a bounded sample of the workload per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # cold row + a few continued rows, sized to ~10 s per step at N = 10^4 on 16 cores
    n_rows = 3 if cfg.N >= 5000 else (8 if cfg.N >= 1000 else min(num_phi, 200))
    rows = list(range(num_phi // 2, num_phi // 2 + n_rows))
    for _ in range(args.warmup):
        oracle_sample(cfg, rows[:1] if cfg.N >= 5000 else rows, num_phi)
    t_all, roots_all, cores = 0.0, 0, 1
    for _ in range(args.steps):
        dt, nroots, cores = oracle_sample(cfg, rows, num_phi)
        t_all += dt
        roots_all += nroots
    value = roots_all / t_all
    sample = (f"per step: rows {rows[0]}..{rows[-1]} of {num_phi} (first cold-started from z_i+/-1, the rest continued) "
              f"+ their caustic points")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_all / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg.name}: N={cfg.N}, num_phi={num_phi} (bounded sample)", "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    args = parse()
    cfg = CONFIGS[args.workload]
    num_phi = args.num_phi or cfg.num_phi
    if args.impl == "reference":
        run_reference(args, cfg, num_phi)
        return

    import torch
    import torch.distributed as dist
    from paper_2506_02121_b200 import api

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    api.lib()
    n_r = 2 * cfg.N
    from paper_2506_02121_b200 import sharding
    phi_off, phi_total = sharding.phase_shard(rank, world, num_phi)
    opt = api.options(num_subchains=args.subchains, predictor_order=args.order, min_lanes_per_root=args.min_lanes,
                      phi_index_offset=phi_off, phi_index_total=phi_total,
                      aberth_sum_precision=args.aberth_sum, skip_aberth_sum_below=args.skip_aberth_below,
                      star_sum_mode=api.MLCC_STAR_SUMS_FMM if args.star_sums == "fmm" else api.MLCC_STAR_SUMS_DIRECT,
                      trust_predictor=1 if args.trust_predictor else 0)

    roots = torch.empty((num_phi, n_r, 2), dtype=torch.float64, device="cuda")
    prev = torch.empty_like(roots)
    caus = torch.empty_like(roots)
    last = {}

    def step():
        xy, m, R = api.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
        if args.separate_caustics:
            _, _, _, st = api.critical_curves_ex(xy, m, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter,
                                                 opt=opt, out_roots=roots, want_diagnostics=False)
            api.caustics(xy, m, cfg.kappa_s, cfg.gamma, roots, out=caus)
        else:
            _, _, _, _, st = api.curves_and_caustics(xy, m, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter,
                                                     opt=opt, out_roots=roots, out_caustics=caus,
                                                     want_diagnostics=False)
        # the very first call has no previous step to compare with (`prev` is uninitialised memory, for which the
        # matcher falls back to its O(n^2) search): it checks the sets against themselves
        err, bij = api.match_root_sets(roots, prev if last else roots, 1e-10)
        v1, v2 = api.vieta_residuals(xy, m, cfg.kappa_s, cfg.gamma, roots, phi_off, phi_total)   # completeness of every row
        last.update(stats=st, err=err, bij=bij, v1=v1, v2=v2)
        return st

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # The clock sampler is started BEFORE the warm-up: nvidia-smi takes a few hundred ms to attach to the driver, and
    # while it does, kernel launches of this process can stall (seen as 100-200 ms added to one timed step).  Only the
    # samples that arrive inside the timed region are reported.
    sampler = ClockSampler(local_rank, args.clock_sample_ms)
    if rank == 0 and args.clock_sample_ms > 0:
        sampler.start()
    # warm-up (also fills `prev` for the validator)
    for w in range(max(args.warmup, 1)):
        step()
        prev.copy_(roots)
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    solve_ms = 0.0
    launches = 0
    alg_flop = 0.0
    alg_flop_survey = 0.0
    compute_launches = 0
    barrier()
    t_begin = time.time()
    ev0.record()
    for _ in range(args.steps):
        st = step()
        solve_ms += st.solve_ms
        launches += st.kernel_launches + 3 + 1 + 2 + (1 if args.separate_caustics else 0)   # star field (3), matcher, Vieta sums (2), caustics
        # root-iterations without the Aberth sum take the Newton step of F and do not accumulate S1 either
        # (R27): their star pairs are 2 flop (one complex addition) lighter
        iters_without_A = st.root_iterations - st.root_pairs / float(n_r - 1)
        alg_flop += (0.0 if args.star_sums == "fmm" else
                     FLOP_PER_STAR_PAIR * st.star_pairs - 2.0 * cfg.N * iters_without_A) + FLOP_PER_ROOT_PAIR * st.root_pairs
        alg_flop_survey += (FLOP_PER_STAR_PAIR * cfg.N + FLOP_PER_ROOT_PAIR * (n_r - 1)) * st.root_iterations
        compute_launches += st.total_iterations
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.stop(t_begin, time.time()) if rank == 0 else None
    st = last["stats"]
    assert bool(last["bij"].all()), "validator: this step's root sets differ from the previous step's"
    assert float(last["v1"].max()) < 1e-12 and float(last["v2"].max()) < 1e-12, "validator: a row fails Vieta's sums"
    assert st.unconverged_rows == 0 and st.degenerate_roots == 0
    t = torch.tensor([ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_max = float(t.item())
    ms_per_step = ms_max / args.steps
    value = world * num_phi * n_r / (ms_per_step * 1e-3)

    # ---- roofline of the dominant kernel (the Aberth compute kernel): FP64 ALU bound ----
    peak_measured = api.fp64_peak(50.0) if rank == 0 else 0.0
    achieved = alg_flop / (solve_ms * 1e-3) / 1e12 if solve_ms > 0 else 0.0
    roofline = {"bound": "alu", "kernel": "mlcc::k_compute (Aberth iteration)", "achieved": achieved,
                "peak": peak_measured, "unit": "TFLOP/s", "frac": achieved / peak_measured if peak_measured else None,
                "peak_source": "measured on this GPU by mlcc_fp64_peak (dependent-free DFMA loop); "
                               f"nominal {NOMINAL_FP64_TFLOPS:.1f} TFLOP/s = 148 SMs x 64 lanes x 2 x 1.965 GHz",
                "frac_of_nominal": achieved / NOMINAL_FP64_TFLOPS,
                "frac_with_survey_accounting": (alg_flop_survey / (solve_ms * 1e-3) / 1e12 / peak_measured
                                                if (solve_ms > 0 and peak_measured and args.star_sums == "direct") else None),
                "algorithmic_flop_per_launch": alg_flop / max(compute_launches, 1),
                "avg_launch_ms": solve_ms / max(compute_launches, 1),
                "note": "achieved = (27 flop x star pairs (25 where S1 is not needed) + 10 flop x root pairs EVALUATED) / device time of the whole solve "
                        "(seed/apply/finalize launches included), CUDA events on the launch stream. Confirming iterations "
                        "of nearly converged roots leave the Aberth sum out (DESIGN.md R27) and their root pairs are not "
                        "counted; frac_with_survey_accounting counts 47N flop for every root-iteration as SURVEY.md 8(d) does",
                # dram__bytes_read.sum + dram__bytes_write.sum of one full-iteration launch of the cfg4 direct-sum kernel
                # (16 rows x 20 000 roots, 1.504e11 algorithmic flop, 6.98 ms) from the ncu --set full capture summarised
                # in profiles/r01_k_compute_ncu.md C: 11.93 MB read, < 0.01 MB written; not measured for other workloads
                "traffic": (NCU_DRAM_BYTES_FULL_ITERATION if (args.workload == "cfg4" and args.star_sums == "direct")
                            else None),
                "traffic_note": "bytes of DRAM traffic per full-iteration launch (ncu capture, profiles/r01_k_compute_ncu.md): "
                                "the working set is L2-resident, 12.6 kflop per DRAM byte; the bound is the ALU one"}

    # ---- measured issue model behind the roofline ----
    if rank == 0:
        probes = {name: api.fp64_issue_probe(form, 20.0) for form, name in
                  ((1, "dfma_3_distinct_sources"), (2, "dadd_2_sources"), (3, "dfma_2_sources_interleaved_with_ffma2"))}
        roofline["issue_model"] = {"unit": "2 x FP64 instructions/s / 1e12", "dfma_2_sources (= peak)": peak_measured,
                                   **probes,
                                   "reading": "one 64-bit register operand per clock per SM sub-partition feeds all pipes: "
                                              "a 3-source DFMA takes 3 clk, and packed FP32 FMAs take operand slots away "
                                              "from the FP64 stream"}

    # ---- post-processing of the timed step's outputs, outside the timed region ----
    post = None
    if args.post and world == 1:
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
        post = {"unit": "ms per call (best of 3, CUDA events)", "rows": num_phi, "roots_per_row": n_r,
                "map": f"{n_pix} x {n_pix} pixels of {pixel:.4f} theta_star",
                "link_rows": t_link, "rows_not_bijective": int((lbij == 0).sum()),
                "closed_loops": t_loops, "num_loops": int(cnt.item()), "chains_not_closed": int((lid < 0).sum()),
                "order_by_chain": t_order, "order_by_chain_GBps": gather_bytes / t_order / 1e6,
                "crossing_map": t_cross, "max_crossings": int(cmap.max()),
                "distance_map": t_edt, "directional_distance_map_(0,1)": t_dir,
                "rays_that_met_a_caustic": float((ddir > 0).double().mean())}
        del nxt, col, cmap, dmap, ddir

    # ---- the same workload with the paper's far-field split of the star sums, outside the timed region ----
    far_field = None
    if world == 1 and args.star_sums == "direct" and not args.no_e2e:
        fopt = api.options(num_subchains=args.subchains, predictor_order=args.order, min_lanes_per_root=args.min_lanes,
                           phi_index_offset=phi_off, phi_index_total=phi_total, aberth_sum_precision=args.aberth_sum,
                           skip_aberth_sum_below=args.skip_aberth_below, star_sum_mode=api.MLCC_STAR_SUMS_FMM)
        fxy, fm, _ = api.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
        best = None
        for _ in range(2):
            torch.cuda.synchronize()
            f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            f0.record()
            _, _, _, _, fst = api.curves_and_caustics(fxy, fm, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter,
                                                      opt=fopt, out_roots=caus, out_caustics=prev, want_diagnostics=False)
            f1.record()
            torch.cuda.synchronize()
            t_ms = f0.elapsed_time(f1)
            best = t_ms if best is None or t_ms < best else best
        ferr, fbij = api.match_root_sets(caus, roots, 1e-10)    # far-field roots against the direct ones of the timed steps
        far_field = {"value": num_phi * n_r / (best * 1e-3), "unit": UNIT, "seconds_per_curve_set": best * 1e-3,
                     "matches_direct_root_sets": bool(fbij.all()), "max_abs_dz_vs_direct": float(ferr.max()),
                     "note": "mlcc_options.star_sum_mode = MLCC_STAR_SUMS_FMM: stars of the 5x5 nodes around a root directly, "
                             "the rest from the node's order-31 Taylor series; the Aberth sum over roots stays direct. "
                             "Not the headline: BASELINE.json fixes direct O(N) star sums"}

    # ---- the same workload with mlcc_options.trust_predictor (R30), outside the timed region ----
    predicted = None
    if world == 1 and args.star_sums == "direct" and not args.trust_predictor and not args.no_e2e:
        predicted = {"unit": UNIT,
                     "note": "mlcc_options.trust_predictor = 1: rows seeded by the cubic predictor start with Newton steps "
                             "(no Aberth sum); a step above 1e-8 is discarded and that root gets the full Aberth iteration. "
                             "Cold rows and fallbacks keep Eq. 17. Not the headline: the headline evaluates the Aberth sum "
                             "for every root of every row"}
        for label, mode in (("direct_star_sums", api.MLCC_STAR_SUMS_DIRECT), ("far_field_star_sums", api.MLCC_STAR_SUMS_FMM)):
            topt = api.options(num_subchains=args.subchains, predictor_order=args.order, min_lanes_per_root=args.min_lanes,
                               phi_index_offset=phi_off, phi_index_total=phi_total, aberth_sum_precision=args.aberth_sum,
                               skip_aberth_sum_below=args.skip_aberth_below, star_sum_mode=mode, trust_predictor=1)
            best, tst = None, None
            for _ in range(2):
                torch.cuda.synchronize()
                f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                f0.record()
                _, _, _, _, tst = api.curves_and_caustics(fxy, fm, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter,
                                                          opt=topt, out_roots=caus, out_caustics=prev, want_diagnostics=False)
                f1.record()
                torch.cuda.synchronize()
                t_ms = f0.elapsed_time(f1)
                best = t_ms if best is None or t_ms < best else best
            terr, tbij = api.match_root_sets(caus, roots, 1e-10)
            predicted[label] = {"value": num_phi * n_r / (best * 1e-3), "seconds_per_curve_set": best * 1e-3,
                                "matches_headline_root_sets": bool(tbij.all()), "max_abs_dz_vs_headline": float(terr.max()),
                                "unconverged_rows": tst.unconverged_rows,
                                "root_iterations_per_root": tst.root_iterations / float(num_phi * n_r),
                                "root_iterations_with_aberth_sum_per_root": tst.root_pairs / float(n_r - 1) / float(num_phi * n_r)}

    # ---- end to end through the host-buffer C-ABI call (pinned host memory both ways) ----
    e2e = None
    if not args.no_e2e:
        gxy, gm, _ = api.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
        p_xy = gxy.cpu().pin_memory()     # the user's host arrays (outside the timed region)
        p_m = gm.cpu().pin_memory()
        h_roots = torch.empty((num_phi, n_r, 2), dtype=torch.float64, pin_memory=True)
        h_caus = torch.empty((num_phi, n_r, 2), dtype=torch.float64, pin_memory=True)
        del prev
        torch.cuda.empty_cache()
        api.curves_and_caustics_host(p_xy, p_m, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter, opt=opt,
                                     out_roots=h_roots, out_caustics=h_caus)       # warm-up
        barrier()
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
        e2e = {"value": world * num_phi * n_r / float(te.item()), "unit": UNIT,
               "h2d_bytes_per_step": int(p_xy.numel() * 8 + p_m.numel() * 8),
               "d2h_bytes_per_step": int(h_roots.numel() * 8 + h_caus.numel() * 8),
               "seconds_per_step": float(te.item()),
               "call": "mlcc_curves_and_caustics_host (host pointers; device alloc + H2D + solve + caustics + D2H inside)"}

    # ---- CPU baseline: the oracle as it stands on a bounded sample (rank 0, N = 1 only) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n_rows = 3 if cfg.N >= 5000 else (8 if cfg.N >= 1000 else min(num_phi, 200))
        rows = list(range(num_phi // 2, num_phi // 2 + n_rows))
        dt, nroots, cores = oracle_sample(cfg, rows, num_phi)
        cpu = {"value": nroots / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
               "sample": f"rows {rows[0]}..{rows[-1]} of {num_phi} ({n_rows} phases: first cold-started from z_i+/-1, "
                         f"the rest continued) + their caustic points"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": f"{cfg.name}: N={cfg.N} stars, {num_phi} phases per GPU, kappa_star={cfg.kappa_star}, "
                                       f"kappa_s={cfg.kappa_s}, gamma={cfg.gamma}, tol={cfg.tol}, max_iter={cfg.max_iter}, seed={cfg.seed}",
                           "step": ("star_field + critical_curves_ex + caustics + match_root_sets + vieta_residuals" if args.separate_caustics
                                    else "star_field + curves_and_caustics (fused) + match_root_sets + vieta_residuals"),
                           "aberth_sum_precision": st.aberth_sum_precision, "star_sums": args.star_sums, "trust_predictor": bool(args.trust_predictor),
                           "subchains": st.subchains, "predictor_order": st.predictor_order,
                           "l2": f"inputs larger than L2: each step writes {2 * num_phi * n_r * 16 / 1e9:.2f} GB of roots and caustics "
                                 f"and reads a {num_phi * n_r * 16 / 1e9:.2f} GB comparison set (L2 is 126 MB)",
                           "seconds_per_curve_set": st.solve_ms * 1e-3,
                           "aberth_iterations_per_step": st.total_iterations,
                           "root_iterations_per_root": st.root_iterations / float(num_phi * n_r)},
                "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu,
                "far_field": far_field}
        if post is not None:
            line["post_processing"] = post
        if predicted is not None:
            line["predicted_newton"] = predicted
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
