"""CPU oracle for the hot path of arXiv 2506.02121 — TEST INFRASTRUCTURE ONLY.

numpy-facing wrappers (argument marshalling only) around oracle/liboracle.so, which is
compiled from oracle/mlcc_oracle.c.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from the
product package and the product never imports it.
"""
import ctypes as C

import numpy as np

from .build import build as _build

_lib = None

_d = np.float64
_pd = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_pi32 = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_pi64 = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        L.orc_critical_curves.argtypes = [_pd, _pd, C.c_int64, C.c_double, C.c_double, C.c_int64,
                                          C.c_double, C.c_int, _pd, _pi32, _pi32]
        for f in (L.orc_critical_curve_rows, L.orc_critical_curve_rows_ld):
            f.argtypes = [_pd, _pd, C.c_int64, C.c_double, C.c_double, C.c_int64, C.c_int64,
                          _pi64, C.c_int64, C.c_double, C.c_int, C.c_void_p, _pd, _pi32, _pi32]
        for f in (L.orc_caustics, L.orc_caustics_ld):
            f.argtypes = [_pd, _pd, C.c_int64, C.c_double, C.c_double, _pd, C.c_int64, _pd]
        for f in (L.orc_residuals, L.orc_residuals_ld):
            f.argtypes = [_pd, _pd, C.c_int64, C.c_double, C.c_double, C.c_double, C.c_double,
                          _pd, C.c_int64, _pd]
        for f in (L.orc_star_sums, L.orc_star_sums_ld):
            f.argtypes = [_pd, _pd, C.c_int64, _pd, C.c_int64, _pd]
        L.orc_match_root_sets.argtypes = [_pd, _pd, C.c_int64, C.c_int64, C.c_double, _pd, _pi32]
        L.orc_rect_sheet.argtypes = [C.c_double, C.c_double, C.c_double, C.c_int, _pd, C.c_int64, C.c_void_p,
                                     C.c_void_p, C.c_void_p]
        L.orc_rect_truncation.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, C.c_double]
        L.orc_rect_critical_curve_rows.argtypes = [_pd, _pd, C.c_int64, C.c_double, C.c_double, C.c_double, C.c_double,
                                                   C.c_double, C.c_int, C.c_double, C.c_int64, _pi64, C.c_int64,
                                                   C.c_double, C.c_int, C.c_void_p, _pd, _pi32, _pi32]
        L.orc_rect_caustics.argtypes = [_pd, _pd, C.c_int64, C.c_double, C.c_double, C.c_double, C.c_double,
                                        C.c_double, C.c_int, _pd, C.c_int64, _pd]
        L.orc_link_rows.argtypes = [_pd, C.c_int64, C.c_int64, _pi32, _pi32]
        L.orc_crossing_map.argtypes = [_pd, C.c_void_p, C.c_int64, C.c_int64, C.c_double, C.c_double, C.c_double,
                                       C.c_int32, C.c_int32, _pi32, C.c_void_p]
        L.orc_closed_loops.argtypes = [_pi32, C.c_int64, C.c_int64, C.c_void_p, _pi32, _pi32, _pi32]
        L.orc_distance_map.argtypes = [_pi32, C.c_int32, C.c_int32, C.c_double, _pd, _pi64]
        L.orc_directional_distance_map.argtypes = [_pi32, C.c_int32, C.c_int32, C.c_double, C.c_int32, C.c_int32, _pd]
        L.orc_distance_histogram.argtypes = [_pd, C.c_void_p, C.c_int64, C.c_double, C.c_int32, C.c_int32, _pi64, _pi64]
        L.orc_vieta_residuals.argtypes = [_pd, _pd, C.c_int64, C.c_double, C.c_double, _pd, C.c_int64, C.c_int64,
                                          C.c_int64, _pd, _pd]
        L.orc_star_field.argtypes = [C.c_uint64, C.c_int64, C.c_double, C.c_int, C.c_void_p,
                                     _pd, _pd, C.POINTER(C.c_double)]
        L.orc_star_field_rect.argtypes = [C.c_uint64, C.c_int64, C.c_double, C.c_double, C.c_int, C.c_void_p,
                                          _pd, _pd, _pd]
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32),
                                        C.POINTER(C.c_uint32)]
        L.orc_philox4x32_10.restype = None
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def num_threads() -> int:
    return int(lib().orc_num_threads())


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def star_field(seed, N, kappa_star, mass_model=0, mass_params=None):
    """-> (star_xy [N,2] f64, masses [N] f64, R)."""
    xy = np.empty((N, 2), _d)
    m = np.empty(N, _d)
    R = C.c_double(0.0)
    pp = None
    if mass_params is not None:
        arr = np.ascontiguousarray(mass_params, _d)
        pp = arr.ctypes.data_as(C.c_void_p)
    _check(lib().orc_star_field(int(seed), int(N), float(kappa_star), int(mass_model), pp, xy, m,
                                C.byref(R)), "star_field")
    return xy, m, R.value


def star_field_rect(seed, N, kappa_star, aspect, mass_model=0, mass_params=None):
    """-> (star_xy [N,2] f64, masses [N] f64, c1, c2): stars uniform in the rectangle with corner c1 + i c2."""
    xy = np.empty((N, 2), _d)
    m = np.empty(N, _d)
    c = np.zeros(2, _d)
    pp = None
    if mass_params is not None:
        arr = np.ascontiguousarray(mass_params, _d)
        pp = arr.ctypes.data_as(C.c_void_p)
    _check(lib().orc_star_field_rect(int(seed), int(N), float(kappa_star), float(aspect), int(mass_model), pp, xy, m, c),
           "star_field_rect")
    return xy, m, float(c[0]), float(c[1])


def _stars(star_xy, masses):
    xy = np.ascontiguousarray(star_xy, _d).reshape(-1, 2)
    m = np.ascontiguousarray(masses, _d).reshape(-1)
    assert xy.shape[0] == m.shape[0]
    return xy, m, xy.shape[0]


def critical_curves(star_xy, masses, kappa_s, gamma, num_phi, tol=1e-12, max_iter=50):
    """Sequential continuation over the whole grid. -> (roots [num_phi,2N,2], iters, unconverged)."""
    xy, m, N = _stars(star_xy, masses)
    out = np.empty((num_phi, 2 * N, 2), _d)
    it = np.zeros(num_phi, np.int32)
    un = np.zeros(num_phi, np.int32)
    _check(lib().orc_critical_curves(xy, m, N, float(kappa_s), float(gamma), int(num_phi),
                                     float(tol), int(max_iter), out, it, un), "critical_curves")
    return out, it, un


def critical_curve_rows(star_xy, masses, kappa_s, gamma, num_phi_total, rows, tol=1e-12,
                        max_iter=50, j_offset=0, init_roots=None, long_double=False):
    """Listed rows; first from cold seeds (or init_roots), each next from the previous listed row."""
    xy, m, N = _stars(star_xy, masses)
    rows = np.ascontiguousarray(rows, np.int64)
    out = np.empty((len(rows), 2 * N, 2), _d)
    it = np.zeros(len(rows), np.int32)
    un = np.zeros(len(rows), np.int32)
    ip = None
    if init_roots is not None:
        init = np.ascontiguousarray(init_roots, _d).reshape(2 * N, 2)
        ip = init.ctypes.data_as(C.c_void_p)
    f = lib().orc_critical_curve_rows_ld if long_double else lib().orc_critical_curve_rows
    _check(f(xy, m, N, float(kappa_s), float(gamma), int(num_phi_total), int(j_offset), rows,
             len(rows), float(tol), int(max_iter), ip, out, it, un), "critical_curve_rows")
    return out, it, un


def caustics(star_xy, masses, kappa_s, gamma, points, long_double=False):
    xy, m, N = _stars(star_xy, masses)
    pts = np.ascontiguousarray(points, _d)
    shape = pts.shape
    flat = pts.reshape(-1, 2)
    out = np.empty_like(flat)
    f = lib().orc_caustics_ld if long_double else lib().orc_caustics
    _check(f(xy, m, N, float(kappa_s), float(gamma), flat, flat.shape[0], out), "caustics")
    return out.reshape(shape)


def residuals(star_xy, masses, kappa_s, gamma, phi_index, num_phi_total, points, long_double=True):
    """-> dict(F complex, Fp complex, inv_mu, newton = |F|/|F'|) at the points, phase 2 pi phi_index/num_phi_total."""
    xy, m, N = _stars(star_xy, masses)
    flat = np.ascontiguousarray(points, _d).reshape(-1, 2)
    out = np.empty((flat.shape[0], 6), _d)
    f = lib().orc_residuals_ld if long_double else lib().orc_residuals
    _check(f(xy, m, N, float(kappa_s), float(gamma), float(phi_index), float(num_phi_total), flat,
             flat.shape[0], out), "residuals")
    return {"F": out[:, 0] + 1j * out[:, 1], "Fp": out[:, 2] + 1j * out[:, 3],
            "inv_mu": out[:, 4].copy(), "newton": out[:, 5].copy()}


def vieta_residuals(star_xy, masses, kappa_s, gamma, roots, j_offset=0, num_phi_total=None):
    """roots [num_phi, 2N, 2] -> (e1 [num_phi], e2 [num_phi]): relative defects of Vieta's first two sums per row."""
    xy, m, N = _stars(star_xy, masses)
    r = np.ascontiguousarray(roots, _d)
    assert r.ndim == 3 and r.shape[1] == 2 * N and r.shape[2] == 2
    e1 = np.empty(r.shape[0], _d)
    e2 = np.empty(r.shape[0], _d)
    _check(lib().orc_vieta_residuals(xy, m, N, float(kappa_s), float(gamma), r, r.shape[0], int(j_offset),
                                     int(num_phi_total or r.shape[0]), e1, e2), "vieta_residuals")
    return e1, e2


def star_sums(star_xy, masses, points, long_double=True):
    """-> [P, 8]: Re/Im of S1 = sum 1/(z-z_i), S2 = sum m/(z-z_i)^2, S3 = sum m/(z-z_i)^3, Sm = sum m/(z-z_i)."""
    xy, m, N = _stars(star_xy, masses)
    flat = np.ascontiguousarray(points, _d).reshape(-1, 2)
    out = np.empty((flat.shape[0], 8), _d)
    f = lib().orc_star_sums_ld if long_double else lib().orc_star_sums
    _check(f(xy, m, N, flat, flat.shape[0], out), "star_sums")
    return out


def match_root_sets(a, b, rel_tol):
    """a, b: [S,n,2]. -> (max_err [S], bijective [S])."""
    a = np.ascontiguousarray(a, _d)
    b = np.ascontiguousarray(b, _d)
    assert a.shape == b.shape and a.ndim == 3 and a.shape[2] == 2
    S, n, _ = a.shape
    err = np.empty(S, _d)
    bij = np.empty(S, np.int32)
    _check(lib().orc_match_root_sets(a, b, S, n, float(rel_tol), err, bij), "match_root_sets")
    return err, bij


def link_rows(rows):
    """rows [S,n,2] -> (next [S,n] int32: column of row (s+1) % S that continues column i of row s, bijective [S])."""
    rows = np.ascontiguousarray(rows, _d)
    S, n, _ = rows.shape
    nxt = np.empty((S, n), np.int32)
    bij = np.empty(S, np.int32)
    _check(lib().orc_link_rows(rows, S, n, nxt, bij), "link_rows")
    return nxt, bij


def crossing_map(caustics, nxt, x0, y0, pixel, nx, ny, want_ambiguous=False):
    """caustics [S,n,2], nxt [S,n] int32 or None -> number of caustic crossings per pixel [ny,nx] int32
    (and, if asked, the uint8 mask of pixels whose centre is within rounding of a segment)."""
    caustics = np.ascontiguousarray(caustics, _d)
    S, n, _ = caustics.shape
    out = np.empty((ny, nx), np.int32)
    amb = np.zeros((ny, nx), np.uint8) if want_ambiguous else None
    if nxt is not None:
        nxt = np.ascontiguousarray(nxt, np.int32)
        assert nxt.shape == (S, n)
    _check(lib().orc_crossing_map(caustics, None if nxt is None else nxt.ctypes.data, S, n, float(x0), float(y0),
                                  float(pixel), int(nx), int(ny), out, None if amb is None else amb.ctypes.data),
           "crossing_map")
    return (out, amb) if want_ambiguous else out


def closed_loops(nxt, want_chain_col=True):
    """nxt [S,n] int32 (link_rows) -> dict(chain_col [S,n] or None, chain_end [n], loop_id [n], num_loops)."""
    nxt = np.ascontiguousarray(nxt, np.int32)
    S, n = nxt.shape
    col = np.empty((S, n), np.int32) if want_chain_col else None
    end = np.empty(n, np.int32)
    lid = np.empty(n, np.int32)
    cnt = np.zeros(1, np.int32)
    _check(lib().orc_closed_loops(nxt, S, n, None if col is None else col.ctypes.data, end, lid, cnt), "closed_loops")
    return {"chain_col": col, "chain_end": end, "loop_id": lid, "num_loops": int(cnt[0])}


def distance_map(cmap, pixel):
    """crossing map [ny,nx] int32 -> (distance to the nearest caustic pixel [ny,nx] f64, squared distance in pixels int64)."""
    cmap = np.ascontiguousarray(cmap, np.int32)
    ny, nx = cmap.shape
    out = np.empty((ny, nx), _d)
    d2 = np.empty((ny, nx), np.int64)
    _check(lib().orc_distance_map(cmap, nx, ny, float(pixel), out, d2), "distance_map")
    return out, d2


def directional_distance_map(cmap, pixel, ux, uy):
    """crossing map [ny,nx] int32, integer direction (ux, uy) -> signed distance along the ray [ny,nx] f64
    (negative: the ray left the map first, |value| = distance to the exit point)."""
    cmap = np.ascontiguousarray(cmap, np.int32)
    ny, nx = cmap.shape
    out = np.empty((ny, nx), _d)
    _check(lib().orc_directional_distance_map(cmap, nx, ny, float(pixel), int(ux), int(uy), out),
           "directional_distance_map")
    return out


def distance_histogram(distance, cmap, bin_width, num_bins, num_counts=1):
    """distance map [ny,nx] f64, crossing map [ny,nx] int32 or None -> (hist [num_counts, num_bins] int64, pixels left out)."""
    d = np.ascontiguousarray(distance, _d)
    cm = None if cmap is None else np.ascontiguousarray(cmap, np.int32)
    assert cm is None or cm.shape == d.shape
    hist = np.empty((num_counts, num_bins), np.int64)
    left = np.zeros(1, np.int64)
    _check(lib().orc_distance_histogram(d, None if cm is None else cm.ctypes.data, d.size, float(bin_width), int(num_bins),
                                        int(num_counts), hist, left), "distance_histogram")
    return hist, int(left[0])


def rect_sheet(kappa_star, c1, c2, t, points):
    """Eq. B2, B7, B9 as printed -> (alpha_s, d alpha_s/d zbar, d2 alpha_s/d zbar2) as complex arrays."""
    flat = np.ascontiguousarray(points, _d).reshape(-1, 2)
    a, b, d = (np.empty_like(flat) for _ in range(3))
    _check(lib().orc_rect_sheet(float(kappa_star), float(c1), float(c2), int(t), flat, flat.shape[0],
                                a.ctypes.data, b.ctypes.data, d.ctypes.data), "rect_sheet")
    return a[:, 0] + 1j * a[:, 1], b[:, 0] + 1j * b[:, 1], d[:, 0] + 1j * d[:, 1]


def rect_truncation(kappa_star, c1, c2, s=1.5, eps=1e-9):
    t = lib().orc_rect_truncation(float(kappa_star), float(c1), float(c2), float(s), float(eps))
    if t < 0:
        raise RuntimeError("oracle rect_truncation failed")
    return t


def rect_critical_curve_rows(star_xy, masses, kappa_s, gamma, kappa_star, c1, c2, t, seed_radius, num_phi_total,
                             rows, tol=1e-12, max_iter=50, init_roots=None):
    """-> (roots [len(rows), 2N + t - 1, 2], iters, unconverged) for the rectangular sheet."""
    xy, m, N = _stars(star_xy, masses)
    rows = np.ascontiguousarray(rows, np.int64)
    n_r = 2 * N + t - 1
    out = np.empty((len(rows), n_r, 2), _d)
    it = np.empty(len(rows), np.int32)
    un = np.empty(len(rows), np.int32)
    init = None
    if init_roots is not None:
        init = np.ascontiguousarray(init_roots, _d)
        assert init.shape == (n_r, 2)
    _check(lib().orc_rect_critical_curve_rows(xy, m, N, float(kappa_s), float(gamma), float(kappa_star), float(c1),
                                              float(c2), int(t), float(seed_radius), int(num_phi_total), rows,
                                              len(rows), float(tol), int(max_iter),
                                              None if init is None else init.ctypes.data, out, it, un),
           "rect_critical_curve_rows")
    return out, it, un


def rect_caustics(star_xy, masses, kappa_s, gamma, kappa_star, c1, c2, t, points):
    xy, m, N = _stars(star_xy, masses)
    pts = np.ascontiguousarray(points, _d)
    flat = pts.reshape(-1, 2)
    out = np.empty_like(flat)
    _check(lib().orc_rect_caustics(xy, m, N, float(kappa_s), float(gamma), float(kappa_star), float(c1), float(c2),
                                   int(t), flat, flat.shape[0], out), "rect_caustics")
    return out.reshape(pts.shape)
