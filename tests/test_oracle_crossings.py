"""Pins of the oracle's chain joining and caustic-crossing map against things
other than itself: analytic winding numbers of polygons, the Chang-Refsdal caustic of the paper's orientation
claim, and the image multiplicity of a binary lens counted by solving the lens equation."""
import numpy as np
import pytest

from test_oracle_pins import cplx


def polygon_set(curves):
    """curves: list of complex arrays of equal length S (closed polygons) -> caustics [S, n, 2]."""
    z = np.stack(curves, axis=1)
    return np.stack([z.real, z.imag], axis=2)


def grid_centres(x0, y0, pixel, nx, ny):
    xs = x0 + (np.arange(nx) + 0.5) * pixel
    ys = y0 + (np.arange(ny) + 0.5) * pixel
    return np.meshgrid(xs, ys)


def test_winding_numbers_of_analytic_polygons(orc):
    S = 180
    t = 2 * np.pi * np.arange(S) / S
    cw = np.exp(-1j * t)                       # clockwise unit circle: one crossing inside
    x0 = y0 = -3.05
    pixel, nx, ny = 0.1, 61, 61
    X, Y = grid_centres(x0, y0, pixel, nx, ny)
    r = np.hypot(X, Y)
    sure = (np.abs(r - 1) > 0.01) & (np.abs(r - 2) > 0.01)   # away from the polygons' edges
    m = orc.crossing_map(polygon_set([cw]), None, x0, y0, pixel, nx, ny)
    assert np.array_equal(m[sure], (r < 1).astype(np.int32)[sure])
    m = orc.crossing_map(polygon_set([np.conj(cw)]), None, x0, y0, pixel, nx, ny)      # counter-clockwise: -1
    assert np.array_equal(m[sure], -(r < 1).astype(np.int32)[sure])
    m = orc.crossing_map(polygon_set([cw, 2 * cw]), None, x0, y0, pixel, nx, ny)        # nested: 2 / 1 / 0
    assert np.array_equal(m[sure], ((r < 1).astype(np.int32) + (r < 2))[sure])
    m = orc.crossing_map(polygon_set([cw, 2 * np.conj(cw)]), None, x0, y0, pixel, nx, ny)  # opposite: 0 / -1 / 0
    assert np.array_equal(m[sure], ((r < 1).astype(np.int32) - (r < 2))[sure])
    m = orc.crossing_map(polygon_set([np.exp(-2j * t)]), None, x0, y0, pixel, nx, ny)    # wound twice
    assert np.array_equal(m[sure], 2 * (r < 1).astype(np.int32)[sure])
    # figure of eight x = sin t, y = sin t cos t: the right lobe is traced clockwise (+1), the left one -1
    eight = 2 * (np.sin(t) + 1j * np.sin(t) * np.cos(t))
    m = orc.crossing_map(polygon_set([eight]), None, x0, y0, pixel, nx, ny)
    iy = ny // 2
    assert m[iy, np.searchsorted(X[0], 1.0)] == 1 and m[iy, np.searchsorted(X[0], -1.0)] == -1
    assert m[0, 0] == 0 and set(np.unique(m)) == {-1, 0, 1}
    # area of the unit disc from the pixel count
    m = orc.crossing_map(polygon_set([cw]), None, -1.2, -1.2, 0.01, 240, 240)
    assert abs(m.sum() * 1e-4 - np.pi) < 5e-3


def test_next_table_routes_the_chains(orc):
    """Column order is free from row to row; `next` says where each chain continues.  Shuffling the columns of
    every row and passing the matching table must give the map of the unshuffled polygons; identity must not."""
    rng = np.random.default_rng(4)
    S, n = 90, 5
    t = 2 * np.pi * np.arange(S) / S
    curves = [c + rad * np.exp(-1j * (t + ph)) for c, rad, ph in
              zip([0, 0.5 + 0.5j, -1 - 1j, 1.5, -0.2 + 1.3j], [1.0, 0.7, 0.9, 0.4, 1.4], rng.uniform(0, 6, 5))]
    base = polygon_set(curves)
    perms = np.stack([rng.permutation(n) for _ in range(S)])          # shuffled[s, c] = base[s, perms[s, c]]
    shuffled = np.stack([base[s, perms[s]] for s in range(S)])
    inv = np.argsort(perms, axis=1)
    nxt = np.stack([inv[(s + 1) % S][perms[s]] for s in range(S)]).astype(np.int32)
    ref = orc.crossing_map(base, None, -3, -3, 0.1, 60, 60)
    got = orc.crossing_map(shuffled, nxt, -3, -3, 0.1, 60, 60)
    assert np.array_equal(got, ref) and ref.max() >= 3
    assert not np.array_equal(orc.crossing_map(shuffled, None, -3, -3, 0.1, 60, 60), ref)
    # the oracle's own joining finds that table from the points (chains move by ~0.1 per row, centres are apart)
    far = polygon_set([c * 4 + cplx(base[:, k]) for k, c in enumerate([0, 3 + 3j, -3 - 3j, 6, -1 + 7j])])
    far_sh = np.stack([far[s, perms[s]] for s in range(S)])
    link, bij = orc.link_rows(far_sh)
    assert bij.all() and np.array_equal(link, nxt)


@pytest.mark.parametrize("kappa_s,gamma", [(0.2, 0.35), (0.0, 0.3)])
def test_chang_refsdal_astroid_holds_one_crossing(orc, kappa_s, gamma):
    """One star with gamma < 1 - kappa_s: the caustic is the four-cusped astroid with cusps at +-2 gamma/sqrt(1-kappa_s-gamma)
    on the real axis and +-2 gamma/sqrt(1-kappa_s+gamma) on the imaginary one (tests/golden/chang_refsdal_cusps.txt).
    A source inside it has two more images: the count is 1 inside and 0 outside, with the sign fixed by the paper's
    orientation statement (caustics traced clockwise as phi increases)."""
    xy, m = np.array([[0.0, 0.0]]), np.array([1.0])
    num_phi = 720
    init = np.array([[np.cos(0.3), np.sin(0.3)], [-np.cos(0.3), -np.sin(0.3)]])
    rows = np.arange(num_phi)
    roots, _, un = orc.critical_curve_rows(xy, m, kappa_s, gamma, num_phi, rows, init_roots=init)
    assert un.sum() == 0
    caus = orc.caustics(xy, m, kappa_s, gamma, roots)
    nxt, bij = orc.link_rows(roots)
    assert bij.all()
    cx = 2 * gamma / np.sqrt(1 - kappa_s - gamma)
    cy = 2 * gamma / np.sqrt(1 - kappa_s + gamma)
    n_pix, half = 81, 1.25 * max(cx, cy)
    pixel = 2 * half / n_pix
    mp, amb = orc.crossing_map(caus, nxt, -half, -half, pixel, n_pix, n_pix, want_ambiguous=True)
    X, Y = grid_centres(-half, -half, pixel, n_pix, n_pix)
    c = n_pix // 2
    assert mp[c, c] == 1 and mp[0, 0] == 0 and mp[c, 0] == 0 and set(np.unique(mp)) == {0, 1}
    on_x = mp[c]                                                   # along the real axis: 1 exactly between the cusps
    assert np.array_equal(on_x[np.abs(X[c]) < cx - pixel], np.ones((np.abs(X[c]) < cx - pixel).sum(), np.int32))
    assert not on_x[np.abs(X[c]) > cx + pixel].any()
    on_y = mp[:, c]
    assert on_y[np.abs(Y[:, c]) < cy - pixel].all() and not on_y[np.abs(Y[:, c]) > cy + pixel].any()
    # astroid (x/cx)^(2/3) + (y/cy)^(2/3) = 1
    inside = (np.abs(X) / cx) ** (2 / 3) + (np.abs(Y) / cy) ** (2 / 3)
    sure = np.abs(inside - 1) > 0.08
    assert np.array_equal(mp[sure], (inside < 1).astype(np.int32)[sure])
    # only the row through y = 0 is flagged: the cusps' vertices lie on that scanline to rounding
    assert amb[np.arange(n_pix) != c].sum() <= 4


def count_images(zs, ms, w, lim=3.0, n_seed=48):
    """Images of a point source at w for point masses with no shear: solutions of z - sum m_i/conj(z - z_i) = w,
    by Newton's method on (z, conj z) from a grid of seeds; distinct converged solutions are counted."""
    g = np.linspace(-lim, lim, n_seed)
    z = (g[None, :] + 1j * g[:, None]).ravel() + 0.013 + 0.007j
    with np.errstate(all="ignore"):
        for _ in range(60):
            d = z[:, None] - zs[None, :]
            f = z - (ms[None, :] / np.conj(d)).sum(1) - w
            fzb = (ms[None, :] / np.conj(d) ** 2).sum(1)               # d f / d conj(z)
            den = 1 - np.abs(fzb) ** 2
            step = (f - np.conj(f) * fzb) / den
            step = np.where(np.abs(step) > 0.5, 0.5 * step / np.abs(step), step)
            z = z - step
    d = z[:, None] - zs[None, :]
    res = np.abs(z - (ms[None, :] / np.conj(d)).sum(1) - w)
    good = z[(res < 1e-10) & np.isfinite(res)]
    uniq = []
    for v in good:
        if all(abs(v - u) > 1e-6 for u in uniq):
            uniq.append(v)
    return len(uniq)


def test_crossing_count_predicts_the_image_multiplicity_of_a_binary_lens(orc):
    """Two point masses, no shear or convergence: 3 images outside the caustic, 5 inside (textbook).  In general a
    source gains two images per caustic crossed, so images = 3 + 2 * count: the oracle's whole chain (critical
    curves -> caustic map -> joining -> winding numbers) against a root count of the lens equation itself."""
    zs = np.array([-0.5 + 0j, 0.5 + 0j])
    ms = np.array([0.6, 0.4])
    xy = np.stack([zs.real, zs.imag], axis=1)
    num_phi = 1440
    # cold seeds z_i +- 1 sit on the real axis with the stars (reading R6): start off the axis instead
    init = np.array([[-0.5, 0.9], [0.5, 0.9], [-0.5, -0.9], [0.5, -0.9]])
    roots, _, un = orc.critical_curve_rows(xy, ms, 0.0, 0.0, num_phi, np.arange(num_phi), init_roots=init)
    assert un.sum() == 0
    caus = orc.caustics(xy, ms, 0.0, 0.0, roots)
    nxt, bij = orc.link_rows(roots)
    assert bij.all()
    half, n_pix = 0.9, 13
    pixel = 2 * half / n_pix
    mp, amb = orc.crossing_map(caus, nxt, -half, -half, pixel, n_pix, n_pix, want_ambiguous=True)
    assert mp.max() == 1 and mp.min() == 0 and mp.sum() >= 4
    X, Y = grid_centres(-half, -half, pixel, n_pix, n_pix)
    cz = cplx(caus).ravel()
    checked = 0
    for iy in range(n_pix):
        for ix in range(n_pix):
            w = X[iy, ix] + 1j * Y[iy, ix]
            if np.abs(cz - w).min() < 0.03:      # too close to the caustic for a Newton root count
                continue
            assert count_images(zs, ms, w) == 3 + 2 * mp[iy, ix], (ix, iy, mp[iy, ix])
            checked += 1
    assert checked > 100
