"""Thin Python binding of libmlcc.so (include/mlcc.h): same names, argument marshalling only.

PyTorch supplies device memory (float64 CUDA tensors) and the current stream; every step of the
path runs in the library's own kernels.  There is no CPU fallback: if the library has not been
built, or a tensor is not a contiguous float64 CUDA tensor, the call raises.
"""
import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmlcc.so")

MLCC_OK = 0
MLCC_ERR_INVALID_ARG = 1
MLCC_ERR_CUDA = 2
MLCC_ERR_NOMEM = 3
MLCC_ERR_NOT_CONVERGED = 4
MLCC_ERR_DEGENERATE = 5
MLCC_STAR_SUMS_DIRECT = 0
MLCC_STAR_SUMS_FMM = 1
MLCC_REGIME_AUTO, MLCC_REGIME_TILED, MLCC_REGIME_CHAIN = 0, 1, 2


class MlccError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__(f"{_status_string(status)}: {text}")
        self.status = status


class mlcc_options(C.Structure):
    _fields_ = [("struct_size", C.c_int32), ("num_subchains", C.c_int32),
                ("predictor_order", C.c_int32), ("max_iter_cold", C.c_int32),
                ("phi_index_offset", C.c_int64), ("phi_index_total", C.c_int64),
                ("min_lanes_per_root", C.c_int32), ("aberth_sum_precision", C.c_int32),
                ("star_sum_mode", C.c_int32), ("fmm_order", C.c_int32),
                ("fmm_stars_per_node", C.c_int32), ("trust_predictor", C.c_int32),
                ("sheet_poly", C.c_void_p), ("sheet_poly_n", C.c_int32), ("regime", C.c_int32),
                ("seed_radius", C.c_double), ("skip_aberth_sum_below", C.c_double)]


class mlcc_stats(C.Structure):
    _fields_ = [("root_iterations", C.c_int64), ("star_pairs", C.c_int64), ("root_pairs", C.c_int64),
                ("kernel_launches", C.c_int64), ("total_iterations", C.c_int32), ("steps", C.c_int32),
                ("subchains", C.c_int32), ("predictor_order", C.c_int32),
                ("unconverged_rows", C.c_int32), ("degenerate_roots", C.c_int32),
                ("solve_ms", C.c_float), ("aberth_sum_precision", C.c_int32), ("regime", C.c_int32),
                ("reserved_", C.c_int32)]


@dataclass
class Stats:
    root_iterations: int
    star_pairs: int
    root_pairs: int
    kernel_launches: int
    total_iterations: int
    steps: int
    subchains: int
    predictor_order: int
    unconverged_rows: int
    degenerate_roots: int
    solve_ms: float
    status: int = 0
    aberth_sum_precision: int = 0
    regime: int = 0


_lib = None


def lib() -> C.CDLL:
    """Loads libmlcc.so (built in-tree by paper_2506_02121_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2506_02121_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i64, i32, dbl = C.c_void_p, C.c_int64, C.c_int32, C.c_double
        L.mlcc_version.restype = C.c_int
        L.mlcc_status_string.restype = C.c_char_p
        L.mlcc_status_string.argtypes = [C.c_int]
        L.mlcc_last_error.restype = C.c_char_p
        L.mlcc_options_default.argtypes = [C.POINTER(mlcc_options)]
        L.mlcc_options_default.restype = None
        L.mlcc_star_field.argtypes = [C.c_uint64, i64, dbl, C.c_int, vp, vp, vp, C.POINTER(dbl), vp]
        L.mlcc_star_field_rect.argtypes = [C.c_uint64, i64, dbl, dbl, C.c_int, vp, vp, vp, vp, vp]
        L.mlcc_critical_curves.argtypes = [vp, vp, i64, dbl, dbl, i64, dbl, i32, vp]
        L.mlcc_critical_curves_ex.argtypes = [vp, vp, i64, dbl, dbl, i64, dbl, i32, vp,
                                              C.POINTER(mlcc_options), vp, vp, vp,
                                              C.POINTER(mlcc_stats), vp]
        L.mlcc_curves_and_caustics.argtypes = [vp, vp, i64, dbl, dbl, i64, dbl, i32, vp, vp,
                                               C.POINTER(mlcc_options), vp, vp, vp,
                                               C.POINTER(mlcc_stats), vp]
        L.mlcc_caustics.argtypes = [vp, vp, i64, dbl, dbl, vp, i64, vp, vp]
        L.mlcc_match_root_sets.argtypes = [vp, vp, i64, i64, dbl, vp, vp, vp]
        L.mlcc_match_root_sets_noalloc.argtypes = [vp, vp, i64, i64, dbl, vp, vp, vp]
        L.mlcc_num_roots.restype = C.c_int64
        L.mlcc_num_roots.argtypes = [i64, i32]
        L.mlcc_rect_sheet.argtypes = [dbl, dbl, dbl, dbl, dbl, i32, vp, i32, C.POINTER(dbl)]
        L.mlcc_link_rows.argtypes = [vp, i64, i64, vp, vp, vp]
        L.mlcc_crossing_map.argtypes = [vp, vp, i64, i64, C.c_int, dbl, dbl, dbl, i32, i32, vp, vp]
        L.mlcc_closed_loops.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp]
        L.mlcc_order_by_chain.argtypes = [vp, vp, i64, i64, vp, vp]
        L.mlcc_distance_map.argtypes = [vp, i32, i32, dbl, vp, vp, vp]
        L.mlcc_directional_distance_map.argtypes = [vp, i32, i32, dbl, i32, i32, vp, vp]
        L.mlcc_distance_histogram.argtypes = [vp, vp, i64, dbl, i32, i32, vp, vp, vp]
        L.mlcc_vieta_residuals.argtypes = [vp, vp, i64, dbl, dbl, vp, i64, i64, i64, vp, vp, vp]
        L.mlcc_detj_residuals.argtypes = [vp, vp, i64, dbl, dbl, vp, i64, i64, i64, i64, vp, vp, vp, vp]
        L.mlcc_star_sums.argtypes = [vp, vp, i64, vp, i64, C.c_int, C.c_int, C.c_int, vp, vp]
        L.mlcc_plan_subchains.argtypes = [i64, i64, i32, i32, vp, vp, vp]
        L.mlcc_critical_curves_host.argtypes = [vp, vp, i64, dbl, dbl, i64, dbl, i32, vp]
        L.mlcc_caustics_host.argtypes = [vp, vp, i64, dbl, dbl, vp, i64, vp]
        L.mlcc_curves_and_caustics_host.argtypes = [vp, vp, i64, dbl, dbl, i64, dbl, i32,
                                                    C.POINTER(mlcc_options), vp, vp, C.POINTER(mlcc_stats)]
        L.mlcc_fp64_peak.argtypes = [dbl, C.POINTER(dbl), vp]
        L.mlcc_fp64_issue_probe.argtypes = [C.c_int, dbl, C.POINTER(dbl), vp]
        _lib = L
    return _lib


def _status_string(status: int) -> str:
    return lib().mlcc_status_string(int(status)).decode()


def _raise(status: int):
    raise MlccError(status, lib().mlcc_last_error().decode())


def _dev(t: Optional[torch.Tensor], dtype=torch.float64, name="tensor") -> Optional[int]:
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name} must be a contiguous {dtype} CUDA tensor")
    return t.data_ptr()


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def version() -> int:
    return int(lib().mlcc_version())


def last_error() -> str:
    return lib().mlcc_last_error().decode()


def options(num_subchains=0, predictor_order=-1, max_iter_cold=0, phi_index_offset=0,
            phi_index_total=0, min_lanes_per_root=0, aberth_sum_precision=0, star_sum_mode=0, fmm_order=0,
            fmm_stars_per_node=0, sheet_poly=None, seed_radius=0.0, skip_aberth_sum_below=0.0,
            trust_predictor=0, regime=0) -> mlcc_options:
    o = mlcc_options()
    lib().mlcc_options_default(C.byref(o))
    o.num_subchains = num_subchains
    o.predictor_order = predictor_order
    o.max_iter_cold = max_iter_cold
    o.phi_index_offset = phi_index_offset
    o.phi_index_total = phi_index_total
    o.min_lanes_per_root = min_lanes_per_root
    o.aberth_sum_precision = aberth_sum_precision
    o.star_sum_mode = star_sum_mode
    o.fmm_order = fmm_order
    o.fmm_stars_per_node = fmm_stars_per_node
    o.skip_aberth_sum_below = skip_aberth_sum_below
    o.trust_predictor = int(trust_predictor)
    o.regime = int(regime)
    if sheet_poly is not None:
        arr = np.ascontiguousarray(sheet_poly, np.float64)
        o._keep = arr                       # the struct holds a raw host pointer: keep the array alive
        o.sheet_poly = arr.ctypes.data
        o.sheet_poly_n = int(arr.size)
        o.seed_radius = float(seed_radius)
    return o


def num_roots(N: int, opt=None) -> int:
    """mlcc_num_roots: roots per row (2N, plus deg H' with a sheet polynomial)."""
    return int(lib().mlcc_num_roots(int(N), int(opt.sheet_poly_n) if (opt is not None and opt.sheet_poly) else 0))


def rect_sheet(kappa_star, c1, c2, s=1.5, eps=1e-9, t=0):
    """mlcc_rect_sheet -> (coef [t+1] float64, gamma_shift, t)."""
    coef = np.zeros(512, np.float64)
    shift = C.c_double(0.0)
    tt = lib().mlcc_rect_sheet(float(kappa_star), float(c1), float(c2), float(s), float(eps), int(t),
                               coef.ctypes.data, 512, C.byref(shift))
    if tt < 0:
        _raise(-tt)
    return coef[:tt + 1].copy(), shift.value, tt


def star_field(seed: int, N: int, kappa_star: float, mass_model: int = 0, mass_params=None,
               device="cuda"):
    """mlcc_star_field -> (star_xy [N,2], masses [N], R)."""
    xy = torch.empty((N, 2), dtype=torch.float64, device=device)
    m = torch.empty((N,), dtype=torch.float64, device=device)
    R = C.c_double(0.0)
    pp = None
    if mass_params is not None:
        arr = np.ascontiguousarray(mass_params, np.float64)
        pp = arr.ctypes.data_as(C.c_void_p)
    rc = lib().mlcc_star_field(int(seed), int(N), float(kappa_star), int(mass_model), pp,
                               xy.data_ptr(), m.data_ptr(), C.byref(R), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return xy, m, R.value


def star_field_rect(seed: int, N: int, kappa_star: float, aspect: float, mass_model: int = 0, mass_params=None,
                    device="cuda"):
    """mlcc_star_field_rect -> (star_xy [N,2], masses [N], c1, c2): stars uniform in the rectangle with corner c1 + i c2."""
    xy = torch.empty((N, 2), dtype=torch.float64, device=device)
    m = torch.empty((N,), dtype=torch.float64, device=device)
    corner = np.zeros(2, np.float64)
    pp = None
    if mass_params is not None:
        arr = np.ascontiguousarray(mass_params, np.float64)
        pp = arr.ctypes.data_as(C.c_void_p)
    rc = lib().mlcc_star_field_rect(int(seed), int(N), float(kappa_star), float(aspect), int(mass_model), pp,
                                    xy.data_ptr(), m.data_ptr(), corner.ctypes.data, _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return xy, m, float(corner[0]), float(corner[1])


def critical_curves(star_xy, masses, kappa_s, gamma, num_phi, tol=1e-12, max_iter=50):
    """mlcc_critical_curves (default options, default stream) -> roots [num_phi, 2N, 2]."""
    N = masses.shape[0]
    out = torch.empty((num_phi, 2 * N, 2), dtype=torch.float64, device=masses.device)
    torch.cuda.current_stream().synchronize()  # the call runs on the legacy default stream
    rc = lib().mlcc_critical_curves(_dev(star_xy, name="star_xy"), _dev(masses, name="masses"), N,
                                    float(kappa_s), float(gamma), int(num_phi), float(tol),
                                    int(max_iter), out.data_ptr())
    if rc != MLCC_OK:
        _raise(rc)
    return out


def _stats(st: mlcc_stats, rc: int) -> Stats:
    return Stats(st.root_iterations, st.star_pairs, st.root_pairs, st.kernel_launches,
                 st.total_iterations, st.steps, st.subchains, st.predictor_order,
                 st.unconverged_rows, st.degenerate_roots, st.solve_ms, rc, st.aberth_sum_precision, st.regime)


def critical_curves_ex(star_xy, masses, kappa_s, gamma, num_phi, tol=1e-12, max_iter=50, opt=None,
                       init_roots=None, out_roots=None, want_diagnostics=True, strict=True):
    """mlcc_critical_curves_ex -> (roots [num_phi,2N,2], iters [num_phi] i32, unconverged [num_phi] i32, Stats).

    strict=False returns the outputs also for MLCC_ERR_NOT_CONVERGED / MLCC_ERR_DEGENERATE
    (Stats.status carries the code)."""
    N = masses.shape[0]
    dev = masses.device
    if out_roots is None:
        out_roots = torch.empty((num_phi, num_roots(N, opt), 2), dtype=torch.float64, device=dev)
    iters = unconv = None
    if want_diagnostics:
        iters = torch.zeros((num_phi,), dtype=torch.int32, device=dev)
        unconv = torch.zeros((num_phi,), dtype=torch.int32, device=dev)
    st = mlcc_stats()
    rc = lib().mlcc_critical_curves_ex(
        _dev(star_xy, name="star_xy"), _dev(masses, name="masses"), N, float(kappa_s), float(gamma),
        int(num_phi), float(tol), int(max_iter), _dev(out_roots, name="out_roots"),
        C.byref(opt) if opt is not None else None, _dev(init_roots, name="init_roots"),
        _dev(iters, torch.int32, "iters"), _dev(unconv, torch.int32, "unconverged"), C.byref(st), _stream())
    if rc != MLCC_OK and (strict or rc not in (MLCC_ERR_NOT_CONVERGED, MLCC_ERR_DEGENERATE)):
        _raise(rc)
    return out_roots, iters, unconv, _stats(st, rc)


def curves_and_caustics(star_xy, masses, kappa_s, gamma, num_phi, tol=1e-12, max_iter=50, opt=None,
                        init_roots=None, out_roots=None, out_caustics=None, want_diagnostics=True, strict=True):
    """mlcc_curves_and_caustics (fused a1-a7) -> (roots, caustics [num_phi,2N,2], iters, unconverged, Stats)."""
    N = masses.shape[0]
    dev = masses.device
    if out_roots is None:
        out_roots = torch.empty((num_phi, num_roots(N, opt), 2), dtype=torch.float64, device=dev)
    if out_caustics is None:
        out_caustics = torch.empty((num_phi, num_roots(N, opt), 2), dtype=torch.float64, device=dev)
    iters = unconv = None
    if want_diagnostics:
        iters = torch.zeros((num_phi,), dtype=torch.int32, device=dev)
        unconv = torch.zeros((num_phi,), dtype=torch.int32, device=dev)
    st = mlcc_stats()
    rc = lib().mlcc_curves_and_caustics(
        _dev(star_xy, name="star_xy"), _dev(masses, name="masses"), N, float(kappa_s), float(gamma),
        int(num_phi), float(tol), int(max_iter), _dev(out_roots, name="out_roots"),
        _dev(out_caustics, name="out_caustics"),
        C.byref(opt) if opt is not None else None, _dev(init_roots, name="init_roots"),
        _dev(iters, torch.int32, "iters"), _dev(unconv, torch.int32, "unconverged"), C.byref(st), _stream())
    if rc != MLCC_OK and (strict or rc not in (MLCC_ERR_NOT_CONVERGED, MLCC_ERR_DEGENERATE)):
        _raise(rc)
    return out_roots, out_caustics, iters, unconv, _stats(st, rc)


def caustics(star_xy, masses, kappa_s, gamma, points, out=None):
    """mlcc_caustics: points [..., 2] -> caustic points of the same shape (asynchronous on the current stream)."""
    N = masses.shape[0]
    P = points.numel() // 2
    if out is None:
        out = torch.empty_like(points)
    rc = lib().mlcc_caustics(_dev(star_xy, name="star_xy"), _dev(masses, name="masses"), N,
                             float(kappa_s), float(gamma), _dev(points, name="points"), P,
                             _dev(out, name="out"), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return out


def vieta_residuals(star_xy, masses, kappa_s, gamma, roots, phi_index_offset=0, phi_index_total=0):
    """mlcc_vieta_residuals: roots [num_phi, 2N, 2] -> (e1 [num_phi], e2 [num_phi]) relative defects of Vieta's sums."""
    N = masses.shape[0]
    if roots.dim() != 3 or roots.shape[1] != 2 * N or roots.shape[2] != 2:
        raise ValueError("roots must be [num_phi, 2N, 2]")
    num_phi = roots.shape[0]
    e1 = torch.empty((num_phi,), dtype=torch.float64, device=roots.device)
    e2 = torch.empty((num_phi,), dtype=torch.float64, device=roots.device)
    rc = lib().mlcc_vieta_residuals(_dev(star_xy, name="star_xy"), _dev(masses, name="masses"), N, float(kappa_s),
                                    float(gamma), _dev(roots, name="roots"), num_phi, int(phi_index_offset),
                                    int(phi_index_total), e1.data_ptr(), e2.data_ptr(), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return e1, e2


def detj_residuals(star_xy, masses, kappa_s, gamma, points, phi_index_offset=0, phi_index_total=0, want_points=False):
    """mlcc_detj_residuals: points [num_phi, n, 2] -> (row_newton [num_phi], row_detj [num_phi], residuals [num_phi, n, 6] or
    None): per row max |F|/|F'| and max |1/mu| / bound; per point Re F, Im F, Re F', Im F', 1/mu, |F|/|F'|."""
    if points.dim() != 3 or points.shape[2] != 2:
        raise ValueError("points must be [num_phi, n, 2]")
    num_phi, n, _ = points.shape
    rn = torch.empty((num_phi,), dtype=torch.float64, device=points.device)
    rd = torch.empty((num_phi,), dtype=torch.float64, device=points.device)
    res = torch.empty((num_phi, n, 6), dtype=torch.float64, device=points.device) if want_points else None
    rc = lib().mlcc_detj_residuals(_dev(star_xy, name="star_xy"), _dev(masses, name="masses"), masses.shape[0],
                                   float(kappa_s), float(gamma), _dev(points, name="points") if num_phi else None,
                                   num_phi, n, int(phi_index_offset), int(phi_index_total),
                                   res.data_ptr() if res is not None else None, rn.data_ptr(), rd.data_ptr(), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return rn, rd, res


def link_rows(rows):
    """mlcc_link_rows: rows [S,n,2] -> (next [S,n] i32, bijective [S] i32)."""
    if rows.dim() != 3 or rows.shape[2] != 2:
        raise ValueError("rows must be [S, n, 2]")
    S, n, _ = rows.shape
    nxt = torch.empty((S, n), dtype=torch.int32, device=rows.device)
    bij = torch.empty((S,), dtype=torch.int32, device=rows.device)
    rc = lib().mlcc_link_rows(_dev(rows, name="rows"), S, n, nxt.data_ptr(), bij.data_ptr(), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return nxt, bij


def crossing_map(caustics, nxt, x0, y0, pixel, nx, ny, closed=True):
    """mlcc_crossing_map: caustics [S,n,2], nxt [S,n] i32 or None -> number of caustic crossings [ny,nx] i32."""
    if caustics.dim() != 3 or caustics.shape[2] != 2:
        raise ValueError("caustics must be [S, n, 2]")
    S, n, _ = caustics.shape
    if nxt is not None and tuple(nxt.shape) != (S, n):
        raise ValueError("nxt must be [S, n]")
    out = torch.empty((ny, nx), dtype=torch.int32, device=caustics.device)
    rc = lib().mlcc_crossing_map(_dev(caustics, name="caustics"), _dev(nxt, torch.int32, "nxt"), S, n,
                                 1 if closed else 0, float(x0), float(y0), float(pixel), int(nx), int(ny),
                                 out.data_ptr(), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return out


def closed_loops(nxt, want_chain_col=True):
    """mlcc_closed_loops: nxt [S,n] i32 -> (chain_col [S,n] i32 or None, chain_end [n] i32, loop_id [n] i32,
    num_loops [1] i32), all on the device."""
    if nxt.dim() != 2:
        raise ValueError("nxt must be [S, n]")
    S, n = nxt.shape
    dev = nxt.device
    col = torch.empty((S, n), dtype=torch.int32, device=dev) if want_chain_col else None
    end = torch.empty((n,), dtype=torch.int32, device=dev)
    lid = torch.empty((n,), dtype=torch.int32, device=dev)
    cnt = torch.empty((1,), dtype=torch.int32, device=dev)
    rc = lib().mlcc_closed_loops(_dev(nxt, torch.int32, "nxt"), S, n, None if col is None else col.data_ptr(),
                                 end.data_ptr(), lid.data_ptr(), cnt.data_ptr(), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return col, end, lid, cnt


def order_by_chain(points, chain_col):
    """mlcc_order_by_chain: points [S,n,2], chain_col [S,n] i32 -> [S,n,2] with column k = chain k."""
    if points.dim() != 3 or points.shape[2] != 2 or tuple(chain_col.shape) != tuple(points.shape[:2]):
        raise ValueError("points must be [S, n, 2] and chain_col [S, n]")
    S, n, _ = points.shape
    out = torch.empty_like(points)
    rc = lib().mlcc_order_by_chain(_dev(points, name="points"), _dev(chain_col, torch.int32, "chain_col"), S, n,
                                   out.data_ptr(), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return out


def distance_map(cmap, pixel, want_d2=False):
    """mlcc_distance_map: crossing map [ny,nx] i32 -> distance to the nearest caustic pixel [ny,nx] f64
    (and the exact squared distance in pixels, i64, if asked)."""
    if cmap.dim() != 2:
        raise ValueError("cmap must be [ny, nx]")
    ny, nx = cmap.shape
    out = torch.empty((ny, nx), dtype=torch.float64, device=cmap.device)
    d2 = torch.empty((ny, nx), dtype=torch.int64, device=cmap.device) if want_d2 else None
    rc = lib().mlcc_distance_map(_dev(cmap, torch.int32, "cmap"), nx, ny, float(pixel), out.data_ptr(),
                                 None if d2 is None else d2.data_ptr(), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return (out, d2) if want_d2 else out


def directional_distance_map(cmap, pixel, ux, uy):
    """mlcc_directional_distance_map: crossing map [ny,nx] i32, integer direction -> signed distance [ny,nx] f64."""
    if cmap.dim() != 2:
        raise ValueError("cmap must be [ny, nx]")
    ny, nx = cmap.shape
    out = torch.empty((ny, nx), dtype=torch.float64, device=cmap.device)
    rc = lib().mlcc_directional_distance_map(_dev(cmap, torch.int32, "cmap"), nx, ny, float(pixel), int(ux), int(uy),
                                             out.data_ptr(), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return out


def distance_histogram(distance, cmap, bin_width, num_bins, num_counts=1):
    """mlcc_distance_histogram: distance map f64, crossing map i32 or None (same shape) ->
    (hist [num_counts, num_bins] i64, left_out [1] i64) on the device."""
    if cmap is not None and tuple(cmap.shape) != tuple(distance.shape):
        raise ValueError("cmap must have the shape of distance")
    hist = torch.empty((num_counts, num_bins), dtype=torch.int64, device=distance.device)
    left = torch.empty((1,), dtype=torch.int64, device=distance.device)
    rc = lib().mlcc_distance_histogram(_dev(distance, name="distance"), _dev(cmap, torch.int32, "cmap"),
                                       distance.numel(), float(bin_width), int(num_bins), int(num_counts),
                                       hist.data_ptr(), left.data_ptr(), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return hist, left


def star_sums(star_xy, masses, points, mode=MLCC_STAR_SUMS_DIRECT, fmm_order=0, fmm_stars_per_node=0):
    """mlcc_star_sums: points [P, 2] -> [P, 8] = (S1, S2, S3, Sm) as (re, im) pairs (asynchronous on the current stream)."""
    N = masses.shape[0]
    P = points.numel() // 2
    out = torch.empty((P, 8), dtype=torch.float64, device=masses.device)
    rc = lib().mlcc_star_sums(_dev(star_xy, name="star_xy"), _dev(masses, name="masses"), N,
                              _dev(points, name="points"), P, int(mode), int(fmm_order), int(fmm_stars_per_node),
                              out.data_ptr(), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return out


def match_root_sets(a, b, rel_tol):
    """mlcc_match_root_sets: a, b [S,n,2] -> (max_err [S] f64, bijective [S] i32)."""
    if a.shape != b.shape or a.dim() != 3 or a.shape[2] != 2:
        raise ValueError("a and b must both be [S, n, 2]")
    S, n, _ = a.shape
    err = torch.empty((S,), dtype=torch.float64, device=a.device)
    bij = torch.empty((S,), dtype=torch.int32, device=a.device)
    rc = lib().mlcc_match_root_sets(_dev(a, name="a"), _dev(b, name="b"), S, n, float(rel_tol),
                                    err.data_ptr(), bij.data_ptr(), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return err, bij


def match_root_sets_noalloc(a, b, rel_tol, out_max_err, out_bijective):
    """mlcc_match_root_sets_noalloc: as match_root_sets, but neither this wrapper nor the library allocates: the caller
    passes the outputs (max_err [S] f64, bijective [S] i32).  n <= 8192 points per set."""
    if a.shape != b.shape or a.dim() != 3 or a.shape[2] != 2:
        raise ValueError("a and b must both be [S, n, 2]")
    S, n, _ = a.shape
    if tuple(out_max_err.shape) != (S,) or tuple(out_bijective.shape) != (S,):
        raise ValueError("out_max_err and out_bijective must be [S]")
    rc = lib().mlcc_match_root_sets_noalloc(_dev(a, name="a"), _dev(b, name="b"), S, n, float(rel_tol),
                                            _dev(out_max_err, name="out_max_err"),
                                            _dev(out_bijective, torch.int32, "out_bijective"), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return out_max_err, out_bijective


def plan_subchains(N: int, num_phi: int, num_subchains: int = 0):
    """mlcc_plan_subchains (host only, no CUDA) -> (first_row, centre_row, end_row) int64 arrays."""
    cap = 1024
    f = np.zeros(cap, np.int64)
    c = np.zeros(cap, np.int64)
    e = np.zeros(cap, np.int64)
    n = lib().mlcc_plan_subchains(int(N), int(num_phi), int(num_subchains), cap,
                                  f.ctypes.data, c.ctypes.data, e.ctypes.data)
    if n < 0:
        raise MlccError(-n, "mlcc_plan_subchains")
    return f[:n].copy(), c[:n].copy(), e[:n].copy()


def curves_and_caustics_host(star_xy: np.ndarray, masses: np.ndarray, kappa_s, gamma, num_phi,
                             tol=1e-12, max_iter=50, opt=None, out_roots=None, out_caustics=None,
                             want_caustics=True):
    """mlcc_curves_and_caustics_host: HOST arrays in, HOST arrays out (numpy or pinned torch CPU tensors)."""
    def hptr(x):
        if isinstance(x, torch.Tensor):
            assert not x.is_cuda and x.dtype == torch.float64 and x.is_contiguous()
            return x.data_ptr()
        assert x.dtype == np.float64 and x.flags["C_CONTIGUOUS"]
        return x.ctypes.data
    N = int(masses.shape[0])
    if out_roots is None:
        out_roots = np.empty((num_phi, num_roots(N, opt), 2), np.float64)
    if want_caustics and out_caustics is None:
        out_caustics = np.empty((num_phi, num_roots(N, opt), 2), np.float64)
    st = mlcc_stats()
    rc = lib().mlcc_curves_and_caustics_host(hptr(star_xy), hptr(masses), N, float(kappa_s), float(gamma),
                                             int(num_phi), float(tol), int(max_iter),
                                             C.byref(opt) if opt is not None else None, hptr(out_roots),
                                             hptr(out_caustics) if want_caustics else None, C.byref(st))
    if rc != MLCC_OK:
        _raise(rc)
    return out_roots, out_caustics, _stats(st, rc)


def critical_curves_host(star_xy: np.ndarray, masses: np.ndarray, kappa_s, gamma, num_phi, tol=1e-12, max_iter=50):
    N = int(masses.shape[0])
    out = np.empty((num_phi, 2 * N, 2), np.float64)
    rc = lib().mlcc_critical_curves_host(star_xy.ctypes.data, masses.ctypes.data, N, float(kappa_s),
                                         float(gamma), int(num_phi), float(tol), int(max_iter), out.ctypes.data)
    if rc != MLCC_OK:
        _raise(rc)
    return out


def caustics_host(star_xy: np.ndarray, masses: np.ndarray, kappa_s, gamma, points: np.ndarray):
    N = int(masses.shape[0])
    pts = np.ascontiguousarray(points, np.float64)
    out = np.empty_like(pts)
    rc = lib().mlcc_caustics_host(star_xy.ctypes.data, masses.ctypes.data, N, float(kappa_s), float(gamma),
                                  pts.ctypes.data, pts.size // 2, out.ctypes.data)
    if rc != MLCC_OK:
        _raise(rc)
    return out


def fp64_issue_probe(form: int, ms_target: float = 20.0) -> float:
    """mlcc_fp64_issue_probe: 2 x FP64 instructions/s / 1e12 of operand form 0..3 (see include/mlcc.h)."""
    v = C.c_double(0.0)
    rc = lib().mlcc_fp64_issue_probe(int(form), float(ms_target), C.byref(v), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return v.value


def fp64_peak(ms_target: float = 50.0) -> float:
    """mlcc_fp64_peak: measured DFMA rate in TFLOP/s."""
    v = C.c_double(0.0)
    rc = lib().mlcc_fp64_peak(float(ms_target), C.byref(v), _stream())
    if rc != MLCC_OK:
        _raise(rc)
    return v.value
