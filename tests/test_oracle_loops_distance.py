"""Pins of the oracle's closed-loop extraction (fn. 5 at :217) and of its two distance maps
(Fig. 5) against things other than itself: the chain structure of the Einstein ring and of the
Chang-Refsdal lens, the three textbook topologies of the equal-mass binary lens, permutations with cycles known by
construction, scipy's Euclidean distance transform, a disc, and rays worked out by hand."""
import numpy as np
import pytest

from test_oracle_pins import cplx


# ----------------------------------------------------------------------------------------- closed loops

def loops_of(orc, xy, m, kappa_s, gamma, num_phi, init):
    roots, _, un = orc.critical_curve_rows(xy, m, kappa_s, gamma, num_phi, np.arange(num_phi), init_roots=init,
                                           max_iter=400)      # hand-made seeds far from the roots: a long cold start
    assert un.sum() == 0
    nxt, bij = orc.link_rows(roots)
    assert bij.all()
    return roots, nxt, orc.closed_loops(nxt)


def test_einstein_ring_is_one_loop_of_two_chains(orc):
    """One star, no shear: the roots are +-e^{i phi/2} (SURVEY.md pin P1), so after a whole turn of phi each chain
    has covered half of the ring and arrives where the other one started: "the start of one chain is the end
    of another"."""
    xy, m = np.array([[0.0, 0.0]]), np.array([1.0])
    init = np.array([[np.cos(0.3), np.sin(0.3)], [-np.cos(0.3), -np.sin(0.3)]])
    roots, nxt, lp = loops_of(orc, xy, m, 0.0, 0.0, 360, init)
    assert lp["num_loops"] == 1
    assert np.array_equal(lp["chain_end"], [1, 0]) and np.array_equal(lp["loop_id"], [0, 0])
    # in chain order every column moves continuously: 2 pi / 360 / 2 per row along the unit circle
    z = cplx(roots)
    zc = np.take_along_axis(z, lp["chain_col"], axis=1)
    step = np.abs(np.diff(zc, axis=0))
    assert np.allclose(step, 2 * np.sin(np.pi / 360 / 2), rtol=1e-9)


@pytest.mark.parametrize("kappa_s,gamma,loops", [(0.2, 0.35, 1), (0.0, 0.3, 1), (0.5, 0.55, 2), (0.3, 0.9, 2)])
def test_chang_refsdal_loop_count(orc, kappa_s, gamma, loops):
    """One star with shear: z^2 = m / c(phi), c = (1 - kappa_s) e^{-i phi} - gamma (SURVEY.md pin P2).  c(phi) winds
    once around 0 if gamma < 1 - kappa_s: the square root changes sign over a turn and the two chains join into ONE
    loop (the Chang-Refsdal oval).  If gamma > 1 - kappa_s it does not wind: each chain closes on itself, TWO loops
    (the two separate ovals of the over-focused case)."""
    xy, m = np.array([[0.0, 0.0]]), np.array([1.0])
    init = np.array([[0.8, 0.6], [-0.8, -0.6]])
    _, _, lp = loops_of(orc, xy, m, kappa_s, gamma, 720, init)
    assert lp["num_loops"] == loops
    if loops == 1:
        assert np.array_equal(lp["chain_end"], [1, 0])
    else:
        assert np.array_equal(lp["chain_end"], [0, 1]) and np.array_equal(lp["loop_id"], [0, 1])


@pytest.mark.parametrize("a,loops", [(0.4, 3), (0.45, 3), (0.55, 1), (1.0, 1), (1.35, 1), (1.5, 2), (2.0, 2)])
def test_equal_mass_binary_topologies(orc, a, loops):
    """Two unit masses at +-a, no shear (SURVEY.md pin P3).  The critical curve of a binary lens has three
    topologies (Schneider & Weiss 1986; Erdl & Schneider 1993): for mass ratio 1 the transitions are at separations
    d_c = 2^(-1/2) and d_w = 2 in units of the Einstein radius of the total mass, sqrt 2 here, i.e. at half
    separations a = 1/2 and a = sqrt 2: three loops (close), one (intermediate), two (wide)."""
    xy = np.array([[-a, 0.0], [a, 0.0]])
    m = np.array([1.0, 1.0])
    # seeds with no mirror symmetry (reading R6: symmetric seeds of a symmetric lens stay symmetric)
    init = np.array([[-a + 0.23, 0.9], [a - 0.1, 0.71], [-a - 0.13, -0.8], [a + 0.31, -1.02]])
    roots, nxt, lp = loops_of(orc, xy, m, 0.0, 0.0, 2880, init)
    assert lp["num_loops"] == loops
    # every chain belongs to a loop and the labels are the smallest members
    lid = lp["loop_id"]
    assert (lid >= 0).all() and all(lid[l] == l for l in np.unique(lid))
    # chain order is continuous across the wrap as well: the last point of chain k is next to the first of chain_end[k]
    z = cplx(roots)
    zc = np.take_along_axis(z, lp["chain_col"], axis=1)
    assert np.abs(np.diff(zc, axis=0)).max() < 0.05
    assert np.abs(zc[-1] - z[0, lp["chain_end"]]).max() < 0.05


def test_loops_of_constructed_permutations(orc):
    """`next` is the identity except in the last row, which holds a permutation made of cycles of chosen lengths,
    and the columns of every row are renamed at random: the loops are those cycles whatever the renaming."""
    rng = np.random.default_rng(11)
    lengths = [1, 1, 2, 3, 5, 8, 13, 1, 30]
    n, S = sum(lengths), 17
    sigma = np.empty(n, np.int64)                    # chain k ends where chain sigma[k] starts
    members, k0 = [], 0
    for L in lengths:
        idx = np.arange(k0, k0 + L)
        sigma[idx] = np.roll(idx, -1)
        members.append(idx)
        k0 += L
    shuffle = rng.permutation(n)                     # chain label -> column of row 0
    ren = [shuffle] + [rng.permutation(n) for _ in range(S - 1)]   # ren[s][chain] = column of chain in row s
    nxt = np.empty((S, n), np.int32)
    for s in range(S - 1):
        nxt[s, ren[s]] = ren[s + 1]
    nxt[S - 1, ren[S - 1]] = ren[0][sigma]
    lp = orc.closed_loops(nxt)
    assert lp["num_loops"] == len(lengths)
    for s in range(S):                               # chain that starts in column ren[0][k] sits in column ren[s][k]
        assert np.array_equal(lp["chain_col"][s, ren[0]], ren[s])
    assert np.array_equal(lp["chain_end"][ren[0]], ren[0][sigma])
    for idx in members:
        cols = ren[0][idx]
        assert (lp["loop_id"][cols] == cols.min()).all()
    # a broken table: the chain that meets the -1, and every chain of its loop, is reported as not closed
    bad = nxt.copy()
    victim = members[5][2]
    bad[7, ren[7][victim]] = -1
    lb = orc.closed_loops(bad)
    assert lb["chain_end"][ren[0][victim]] == -1
    assert (lb["loop_id"][ren[0][members[5]]] == -1).all()
    assert lb["num_loops"] == len(lengths) - 1
    keep = np.setdiff1d(np.arange(n), ren[0][members[5]])
    assert np.array_equal(lb["loop_id"][keep], lp["loop_id"][keep])


# ----------------------------------------------------------------------------------------- distance maps

def blob_map(rng, nx, ny, blobs=6):
    """an integer map with several nested / overlapping regions, like a crossing map"""
    X, Y = np.meshgrid(np.arange(nx), np.arange(ny))
    m = np.zeros((ny, nx), np.int32)
    for _ in range(blobs):
        cx, cy = rng.uniform(0, nx), rng.uniform(0, ny)
        rx, ry = rng.uniform(1.5, max(nx / 3, 2)), rng.uniform(1.5, max(ny / 3, 2))
        m += (((X - cx) / rx) ** 2 + ((Y - cy) / ry) ** 2 < 1).astype(np.int32)
    return m


def edge_mask(m):
    e = np.zeros(m.shape, bool)
    e[:, 1:] |= m[:, 1:] != m[:, :-1]
    e[:, :-1] |= m[:, 1:] != m[:, :-1]
    e[1:, :] |= m[1:, :] != m[:-1, :]
    e[:-1, :] |= m[1:, :] != m[:-1, :]
    return e


def test_distance_map_is_the_euclidean_distance_transform(orc):
    """The paper computes this map with "a Euclidean distance transform": scipy's exact transform
    of the same caustic-pixel mask is the library routine the oracle's brute force must reduce to."""
    ndi = pytest.importorskip("scipy.ndimage")
    rng = np.random.default_rng(5)
    for nx, ny in [(37, 23), (64, 64), (5, 90)]:
        m = blob_map(rng, nx, ny)
        d, d2 = orc.distance_map(m, 0.25)
        e = edge_mask(m)
        assert e.any()
        ref = ndi.distance_transform_edt(~e)
        assert np.array_equal(d2, np.rint(ref ** 2).astype(np.int64))
        assert np.allclose(d, 0.25 * ref, rtol=1e-15, atol=0)
        assert (d[e] == 0).all() and (d[~e] >= 0.25).all()
    flat = np.full((6, 9), 3, np.int32)                        # no caustic anywhere: +inf, d2 = -1
    d, d2 = orc.distance_map(flat, 1.0)
    assert np.isinf(d).all() and (d2 == -1).all()


def test_distance_map_of_a_disc(orc):
    """A circular caustic of radius r (count 1 inside): the distance of a source at radius rho is |rho - r| up to
    the pixel size."""
    n, pixel, r = 121, 0.05, 1.7
    X, Y = np.meshgrid((np.arange(n) - n // 2) * pixel, (np.arange(n) - n // 2) * pixel)
    rho = np.hypot(X, Y)
    m = (rho < r).astype(np.int32)
    d, _ = orc.distance_map(m, pixel)
    assert np.abs(d - np.abs(rho - r)).max() < 1.5 * pixel
    assert d[n // 2, n // 2] == pytest.approx(r, abs=1.5 * pixel)


def test_directional_distance_by_hand(orc):
    """Rays worked out on paper.  Map 7 x 5 with a 3 x 3 block of ones in columns 2..4, rows 1..3."""
    m = np.zeros((5, 7), np.int32)
    m[1:4, 2:5] = 1
    e = orc.directional_distance_map(m, 1.0, 1, 0)            # moving in +x
    # row 0 never meets the block: leaves through x = 6.5
    assert np.array_equal(e[0], -(6.5 - np.arange(7)))
    # row 2: from column 0 the block's left border is at x = 1.5; inside the block the right border is at 4.5;
    # behind the block the ray leaves the map
    assert np.array_equal(e[2], [1.5, 0.5, 2.5, 1.5, 0.5, -1.5, -0.5])
    w = orc.directional_distance_map(m, 1.0, -1, 0)           # moving in -x: the mirror image
    assert np.array_equal(w[2], e[2][::-1]) and np.array_equal(w[0], e[0][::-1])
    # the length of the direction vector does not matter
    assert np.array_equal(orc.directional_distance_map(m, 1.0, 5, 0), e)
    # the pixel size scales the result
    assert np.array_equal(orc.directional_distance_map(m, 0.125, 1, 0), 0.125 * e)
    dg = orc.directional_distance_map(m, 1.0, 1, 1)           # along the diagonal
    r2 = np.sqrt(2.0)
    # from (0,0): through the corner (0.5,0.5) into pixel (1,1) (count 0), through (1.5,1.5) into (2,2): a one
    assert dg[0, 0] == pytest.approx(1.5 * r2, rel=1e-15)
    # from (1,0): enters (2,1) through its corner (1.5, 0.5)
    assert dg[0, 1] == pytest.approx(0.5 * r2, rel=1e-15)
    # from (0,3): (1,4) is a zero, then out of the map through y = 4.5
    assert dg[3, 0] == pytest.approx(-1.5 * r2, rel=1e-15)
    # from (5,0): the corner (4.5, 0.5)... the ray runs away from the block and leaves through x = 6.5
    assert dg[0, 5] == pytest.approx(-1.5 * r2, rel=1e-15)
    # a ray that only touches a corner of the block does not enter it: from (1,4) along (1,-1) the point (1.5,3.5)
    # is the block's corner, pixel (2,3) is entered through it
    assert orc.directional_distance_map(m, 1.0, 1, -1)[4, 1] == pytest.approx(0.5 * r2, rel=1e-15)
    # from (0,4) along (1,-1): (0.5,3.5) -> pixel (1,3), a zero -> corner (1.5,2.5) -> pixel (2,2), a one
    assert orc.directional_distance_map(m, 1.0, 1, -1)[4, 0] == pytest.approx(1.5 * r2, rel=1e-15)
    # direction (2,1) from (0,0): x = 2t, y = t; enters column 2 (x = 1.5) at t = 0.75 where y = 0.75 is row 1: a one
    assert orc.directional_distance_map(m, 1.0, 2, 1)[0, 0] == pytest.approx(0.75 * np.sqrt(5.0), rel=1e-15)


def test_directional_distance_against_a_sampled_ray(orc):
    """Independent check at random directions: march along the ray in small steps, read the pixel under the
    sample, stop at the first other count.  The marched distance brackets the exact entry point."""
    rng = np.random.default_rng(8)
    nx, ny = 41, 33
    m = blob_map(rng, nx, ny, blobs=5)
    h = 1e-3
    for ux, uy in [(3, 1), (-2, 5), (1, -4), (-7, -3), (0, 1), (0, -1)]:
        d = orc.directional_distance_map(m, 1.0, ux, uy)
        u = np.array([ux, uy]) / np.hypot(ux, uy)
        for _ in range(60):
            px, py = int(rng.integers(nx)), int(rng.integers(ny))
            t, hit = 0.0, None
            while True:
                t += h
                x, y = px + t * u[0], py + t * u[1]
                ix, iy = int(np.floor(x + 0.5)), int(np.floor(y + 0.5))
                if ix < 0 or iy < 0 or ix >= nx or iy >= ny:
                    hit = -t
                    break
                if m[iy, ix] != m[py, px]:
                    hit = t
                    break
            # a ray that clips less than the step off a pixel's corner is seen by the exact rule only
            if np.sign(hit) == np.sign(d[py, px]):
                assert abs(abs(hit) - abs(d[py, px])) < 2 * h, (ux, uy, px, py, hit, d[py, px])
            else:
                assert hit < 0 or abs(d[py, px]) < abs(hit) + 2 * h


def test_distance_histogram_against_numpy_and_a_disc(orc):
    """The statistics of Fig. 6-7 are histograms of the distance maps.  numpy's histogram is the
    library routine; a circular caustic gives a closed form: inside a disc of radius r the area at distance
    [d, d + h) from the rim is pi ((r - d)^2 - (r - d - h)^2)."""
    rng = np.random.default_rng(12)
    d = rng.uniform(0, 5, size=(40, 60))
    d[rng.random(d.shape) < 0.1] *= -1            # border-limited rays
    d[3, 4] = np.inf
    cm = rng.integers(-1, 7, size=d.shape).astype(np.int32)
    h, left = orc.distance_histogram(d, cm, 0.25, 16, 5)
    ok = (d >= 0) & np.isfinite(d) & (d < 4.0)
    assert left == (~ok).sum() and h.sum() == ok.sum()
    rows = np.clip(cm, 0, 4)
    for r in range(5):
        want, _ = np.histogram(d[ok & (rows == r)], bins=16, range=(0, 4.0))
        assert np.array_equal(h[r], want)
    h1, left1 = orc.distance_histogram(d, None, 0.25, 16)
    assert np.array_equal(h1[0], h.sum(0)) and left1 == left
    # disc
    n, pixel, r = 401, 0.01, 1.5
    X, Y = np.meshgrid((np.arange(n) - n // 2) * pixel, (np.arange(n) - n // 2) * pixel)
    rho = np.hypot(X, Y)
    m = (rho < r).astype(np.int32)
    dist, _ = orc.distance_map(m, pixel)
    hist, _ = orc.distance_histogram(dist, m, 0.1, 12, 2)
    edges = 0.1 * np.arange(13)
    area_in = np.pi * ((r - edges[:-1]) ** 2 - (r - edges[1:]) ** 2) / pixel ** 2
    # bins 1..11 of the inside (bin 0 holds the two-pixel-wide caustic band itself)
    assert np.abs(hist[1, 1:12] / area_in[1:12] - 1).max() < 0.06
    area_out = np.pi * ((r + edges[1:]) ** 2 - (r + edges[:-1]) ** 2) / pixel ** 2
    assert np.abs(hist[0, 1:5] / area_out[1:5] - 1).max() < 0.06      # outside, while the rings stay inside the map
