"""CPU-only checks of the product's host side: the C-ABI library loads and exports every symbol
include/mlcc.h declares; status strings; the sub-chain planner (host logic, no CUDA call);
argument validation that is decided before any CUDA call."""
import ctypes as C
import os
import re
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2506_02121_b200 import build
    build.build()
    from paper_2506_02121_b200 import api
    return api.lib()


def declared_symbols():
    inc = os.path.join(ROOT, "include")
    text = "".join(open(os.path.join(inc, f)).read() for f in sorted(os.listdir(inc)) if f.endswith(".h"))
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mlcc_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_symbols()
    assert len(names) >= 12 and "mlcc_critical_curves" in names and "mlcc_caustics" in names
    for n in names:
        assert hasattr(lib, n), n


def test_version_and_status_strings(lib):
    assert lib.mlcc_version() >= 100
    lib.mlcc_status_string.restype = C.c_char_p
    seen = {lib.mlcc_status_string(i).decode() for i in range(6)}
    assert seen == {"MLCC_OK", "MLCC_ERR_INVALID_ARG", "MLCC_ERR_CUDA", "MLCC_ERR_NOMEM",
                    "MLCC_ERR_NOT_CONVERGED", "MLCC_ERR_DEGENERATE"}
    assert lib.mlcc_status_string(99).decode() == "MLCC_ERR_UNKNOWN"


def test_options_default_and_struct_layout(lib):
    from paper_2506_02121_b200 import api
    o = api.options()
    assert o.struct_size == C.sizeof(api.mlcc_options) == 88
    assert o.predictor_order == -1 and o.num_subchains == 0 and o.phi_index_total == 0
    assert C.sizeof(api.mlcc_stats) == 72


@pytest.mark.parametrize("N,num_phi,req", [(10, 1000, 0), (200, 4000, 0), (2000, 5000, 0), (10000, 10000, 0),
                                           (50000, 2000, 0), (3, 1, 0), (3, 7, 5), (5, 100, 7), (1, 2, 64)])
def test_plan_subchains_covers_every_row_once(lib, N, num_phi, req):
    from paper_2506_02121_b200 import api
    first, centre, end = api.plan_subchains(N, num_phi, req)
    n = len(first)
    assert 1 <= n <= min(num_phi, 512)
    if req:
        assert n == min(req, num_phi)
    assert first[0] == 0 and end[-1] == num_phi
    assert np.all(first[1:] == end[:-1])          # contiguous, disjoint
    assert np.all(end > first)                     # non-empty
    assert np.all((centre >= first) & (centre < end))
    # growing outwards from the centres reaches every row exactly once
    seen = np.zeros(num_phi, int)
    for c in range(n):
        seen[centre[c]] += 1
        s = 1
        while centre[c] - s >= first[c] or centre[c] + s < end[c]:
            if centre[c] - s >= first[c]:
                seen[centre[c] - s] += 1
            if centre[c] + s < end[c]:
                seen[centre[c] + s] += 1
            s += 1
    assert np.all(seen == 1)


def test_plan_subchains_rejects_bad_arguments(lib):
    from paper_2506_02121_b200 import api
    with pytest.raises(api.MlccError):
        api.plan_subchains(0, 10)
    with pytest.raises(api.MlccError):
        api.plan_subchains(5, 0)


def test_invalid_arguments_fail_before_any_cuda_call(lib):
    """Null pointers and out-of-range scalars return MLCC_ERR_INVALID_ARG on a box with no GPU."""
    from paper_2506_02121_b200 import api
    L = lib
    one = 16  # any non-null fake pointer: validation happens before it would be dereferenced
    assert L.mlcc_critical_curves(None, one, 3, 0.0, 0.1, 10, 1e-12, 50, one) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_critical_curves(one, one, 0, 0.0, 0.1, 10, 1e-12, 50, one) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_critical_curves(one, one, 3, 0.0, 0.1, 0, 1e-12, 50, one) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_critical_curves(one, one, 3, 0.0, 0.1, 10, 0.0, 50, one) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_critical_curves(one, one, 3, 0.0, 0.1, 10, 1e-12, 0, one) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_critical_curves(one, one, 3, float("nan"), 0.1, 10, 1e-12, 50, one) == api.MLCC_ERR_INVALID_ARG
    # c(phi_0) = (1 - kappa_s) - gamma = 0: the polynomial's degree drops on row 0
    assert L.mlcc_critical_curves(one, one, 3, 0.5, 0.5, 10, 1e-12, 50, one) == api.MLCC_ERR_INVALID_ARG
    assert b"c(phi_j)" in L.mlcc_last_error()
    assert L.mlcc_caustics(None, one, 3, 0.0, 0.1, one, 5, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_caustics(one, one, 3, 0.0, 0.1, one, -1, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_caustics(one, one, 3, 0.0, 0.1, one, 5, one, None) == api.MLCC_ERR_INVALID_ARG  # aliasing
    assert L.mlcc_caustics(one, one, 3, 0.0, 0.1, None, 0, None, None) == api.MLCC_OK              # P = 0
    assert L.mlcc_match_root_sets(None, one, 2, 5, 1e-10, one, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_match_root_sets(one, one, 2, 0, 1e-10, one, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_match_root_sets(None, None, 0, 5, 1e-10, None, None, None) == api.MLCC_OK       # S = 0
    assert L.mlcc_star_field(0, 0, 0.4, 0, None, one, one, None, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_star_field(0, 5, -1.0, 0, None, one, one, None, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_star_field(0, 5, 0.4, 7, None, one, one, None, None) == api.MLCC_ERR_INVALID_ARG
    L.mlcc_star_field_rect.argtypes = [C.c_uint64, C.c_int64, C.c_double, C.c_double, C.c_int, C.c_void_p, C.c_void_p,
                                       C.c_void_p, C.c_void_p, C.c_void_p]
    assert L.mlcc_star_field_rect(0, 5, 0.4, 0.0, 0, None, one, one, None, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_star_field_rect(0, 5, 0.4, float("inf"), 0, None, one, one, None, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_star_field_rect(0, 0, 0.4, 1.0, 0, None, one, one, None, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_star_field_rect(0, 5, 0.4, 1.0, 0, None, None, one, None, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_fp64_peak(50.0, None, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_star_sums(None, one, 3, one, 5, 0, 0, 0, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_star_sums(one, one, 3, one, 5, 2, 0, 0, one, None) == api.MLCC_ERR_INVALID_ARG   # unknown mode
    assert L.mlcc_star_sums(one, one, 3, one, -1, 0, 0, 0, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_star_sums(one, one, 3, None, 0, 1, 0, 0, None, None) == api.MLCC_OK              # P = 0
    assert L.mlcc_link_rows(None, 3, 5, one, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_link_rows(one, 3, 0, one, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_link_rows(None, 0, 5, None, None, None) == api.MLCC_OK                           # S = 0
    assert L.mlcc_crossing_map(None, None, 3, 5, 1, 0.0, 0.0, 0.1, 8, 8, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_crossing_map(one, None, 3, 5, 1, 0.0, 0.0, 0.0, 8, 8, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_crossing_map(one, None, 3, 5, 1, 0.0, 0.0, 0.1, 0, 8, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_crossing_map(one, None, 0, 5, 1, 0.0, 0.0, 0.1, 8, 8, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_closed_loops(None, 3, 5, None, one, one, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_closed_loops(one, 3, 5, None, None, one, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_closed_loops(one, 0, 5, None, one, one, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_closed_loops(one, 3, 0, None, one, one, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_order_by_chain(None, one, 3, 5, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_order_by_chain(one, one, 3, 5, one, None) == api.MLCC_ERR_INVALID_ARG            # aliasing
    assert L.mlcc_order_by_chain(None, None, 0, 5, None, None) == api.MLCC_OK                      # S = 0
    assert L.mlcc_distance_map(None, 8, 8, 0.1, one, None, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_distance_map(one, 0, 8, 0.1, one, None, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_distance_map(one, 8, 8, -0.1, one, None, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_directional_distance_map(one, 8, 8, 0.1, 0, 0, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_directional_distance_map(one, 8, 8, 0.1, 1 << 21, 1, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_directional_distance_map(one, 8, 8, 0.1, 1, 1, None, None) == api.MLCC_ERR_INVALID_ARG
    L.mlcc_distance_histogram.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_double, C.c_int32, C.c_int32,
                                          C.c_void_p, C.c_void_p, C.c_void_p]
    assert L.mlcc_distance_histogram(one, None, 64, 0.1, 8, 1, None, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_distance_histogram(None, None, 64, 0.1, 8, 1, one, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_distance_histogram(one, None, 64, 0.0, 8, 1, one, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_distance_histogram(one, None, 64, 0.1, 0, 1, one, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_distance_histogram(one, None, 64, 0.1, 1 << 20, 1 << 10, one, one, None) == api.MLCC_ERR_INVALID_ARG
    L.mlcc_vieta_residuals.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_double, C.c_double, C.c_void_p, C.c_int64,
                                       C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
    assert L.mlcc_vieta_residuals(None, one, 3, 0.0, 0.1, one, 4, 0, 0, one, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_vieta_residuals(one, one, 0, 0.0, 0.1, one, 4, 0, 0, one, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_vieta_residuals(one, one, 3, float("nan"), 0.1, one, 4, 0, 0, one, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_vieta_residuals(one, one, 3, 0.0, 0.1, one, 4, 0, 0, None, one, None) == api.MLCC_ERR_INVALID_ARG
    assert L.mlcc_vieta_residuals(one, one, 3, 0.0, 0.1, None, 0, 0, 0, None, None, None) == api.MLCC_OK    # no rows
    o = api.mlcc_options()
    L.mlcc_options_default(C.byref(o))
    assert o.struct_size == C.sizeof(api.mlcc_options) and o.star_sum_mode == api.MLCC_STAR_SUMS_DIRECT


def test_product_does_not_import_the_oracle():
    """The product path may not route through oracle/ (no CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2506_02121_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "liboracle" not in text and "mlcc_oracle" not in text, f
    text = open(os.path.join(ROOT, "include", "mlcc.h")).read()
    assert "oracle" not in text.lower()


def test_rect_sheet_polynomial_reproduces_eq_b2(lib, orc):
    """mlcc_rect_sheet (host-only): its real-coefficient polynomial H and gamma shift against the oracle's literal
    Eq. B2 / B7 (four corners, complex logarithms): alpha_s = -kappa_star z + kappa_star (1 - 4 theta/pi) conj z + H(conj z),
    conj(d alpha_s/d zbar) = -gamma_shift + H'(z); t from Eq. B5 and the (t-1) Arg c rule as the oracle finds it."""
    from paper_2506_02121_b200 import api
    rng = np.random.default_rng(2)
    for kstar, c1, c2 in ((0.4, 3.0, 2.0), (0.25, 2.0, 5.0), (0.6, 4.0, 4.0)):
        coef, shift, t = api.rect_sheet(kstar, c1, c2, s=1.5, eps=1e-9)
        assert t == orc.rect_truncation(kstar, c1, c2, 1.5, 1e-9) and t % 2 == 1 and len(coef) == t + 1
        assert coef[t] != 0.0 and (coef[0::2] == 0).all() and coef[1] == 0
        theta = np.arctan2(c2, c1)
        assert abs(shift + kstar * (1 - 4 * theta / np.pi)) < 1e-15
        pts = rng.uniform(-1, 1, size=(50, 2)) * [c1, c2] * 0.6
        z = pts[:, 0] + 1j * pts[:, 1]
        a, b7, b9 = orc.rect_sheet(kstar, c1, c2, t, pts)
        H = np.polyval(coef[::-1], np.conj(z))
        assert np.abs(-kstar * z - shift * np.conj(z) + H - a).max() < 1e-13
        dH = np.polyval(np.polyder(coef[::-1]), z)
        assert np.abs(-shift + dH - np.conj(b7)).max() < 1e-13
        d2H = np.polyval(np.polyder(coef[::-1], 2), z)
        assert np.abs(d2H - np.conj(b9)).max() < 1e-12
    coef5, _, t5 = api.rect_sheet(0.4, 3.0, 2.0, t=4)          # even request -> odd
    assert t5 % 2 == 1 and t5 >= 5
    assert api.num_roots(7) == 14 and api.num_roots(7, api.options(sheet_poly=coef5, seed_radius=4.0)) == 14 + t5 - 1
    L = lib
    assert L.mlcc_rect_sheet(0.4, -1.0, 2.0, 1.5, 1e-9, 0, coef5.ctypes.data, 6, C.byref(C.c_double())) < 0
    assert L.mlcc_rect_sheet(0.4, 3.0, 2.0, 1.5, 1e-9, 0, coef5.ctypes.data, 6, C.byref(C.c_double())) < 0   # capacity


def test_bench_host_arithmetic():
    """bench.py's host-side bookkeeping (no GPU): the stride of the in-step det J sample reproduces the sampled rows'
    phases exactly, and the per-pipe roofline splits the counters the way the line says it does."""
    import types
    sys.path.insert(0, ROOT)
    import bench
    from paper_2506_02121_b200.configs import CONFIGS
    for total, off in ((10000, 0), (4000, 0), (5000, 0), (2000, 0), (1000, 0), (20000, 10000), (80000, 30000), (7, 0)):
        d = bench.detj_stride(total, off)
        assert 1 <= d <= 64 and total % d == 0 and off % d == 0
        # row q*d of the rank (grid row q*d + off) has phase 2 pi (q + off/d) / (total/d)
        q = 3
        assert abs((q * d + off) / total - (q + off // d) / (total // d)) < 1e-15
    assert bench.detj_stride(10000, 0) == 50
    cfg = CONFIGS["cfg4"]
    n_r = 2 * cfg.N
    st = types.SimpleNamespace(root_iterations=1000, root_pairs=900 * (n_r - 1), aberth_sum_precision=64)
    f64 = bench.flop_model(cfg, st, "direct", 64)
    f32 = bench.flop_model(cfg, st, "direct", 32)
    star = 27.0 * cfg.N * 900 + 25.0 * cfg.N * 100
    assert f64["fp32"] == 0.0 and abs(f64["fp64"] - (star + 10.0 * st.root_pairs)) < 1.0
    assert abs(f32["fp64"] - star) < 1.0 and abs(f32["fp32"] - 10.0 * st.root_pairs) < 1.0
    acc = {"solve_ms": 1000.0, "fp64": f32["fp64"], "fp32": f32["fp32"], "hw_fp64": f32["hw_fp64"], "survey": f32["survey"]}
    rf = bench.roofline_of(acc, 37.0, 70.0, 32)
    assert abs(rf["combined_frac"] - (rf["fp64_frac"] + rf["fp32_frac"])) < 1e-15 and rf["fp32_frac"] > 0
    assert bench.roofline_of(dict(acc, fp32=0.0), 37.0, 70.0, 64)["fp32_frac"] == 0.0


def test_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` (the oracle on the host cores, no GPU): one JSON line with the keys the driver reads,
    the value being the full-set rate extrapolated from a cold row and continued rows, labelled as such."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "cfg1",
                        "--gpus", "1", "--steps", "2", "--warmup", "1"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "converged critical-curve roots/s" and d["unit"] == "roots/s"
    assert d["higher_is_better"] is True and d["n_gpus"] == 1 and d["steps"] == 2 and d["warmup"] == 1
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["vs_baseline"] is None and d["dtype"] == "f64"
    assert d["config"]["workload"].startswith("cfg1") and d["config"]["extrapolated"] is True
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == d["value"] and cb["extrapolated"] is True
    assert cb["seconds_per_cold_row"] > 0 and cb["seconds_per_continued_row"] > 0
    assert abs(cb["extrapolated_full_set_s"] - (cb["seconds_per_cold_row"] + 999 * cb["seconds_per_continued_row"])) < 1e-9
    assert d["e2e"] == {"value": d["value"], "unit": "roots/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["gpu_launches"] == 0
    # ranks other than 0 do no work and print nothing
    r1 = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "cfg1",
                         "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=dict(env, RANK="1", WORLD_SIZE="2"),
                        timeout=300)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
