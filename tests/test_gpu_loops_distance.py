"""GPU parity tests of the chain / closed-loop extraction (mlcc_closed_loops, mlcc_order_by_chain; PAPER.md:209,
fn. 5 at :217) and of the two distance-to-caustic maps (mlcc_distance_map, mlcc_directional_distance_map;
PAPER.md:247, Fig. 5) against the CPU oracle.  Integer outputs are compared exactly; the distances are one square
root / one division away from exact integers and are compared to 1e-15 relative."""
import numpy as np
import pytest

from paper_2506_02121_b200.configs import CONFIGS
from test_oracle_pins import cplx
from test_oracle_loops_distance import blob_map

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2506_02121_b200 import api as a
    a.lib()  # raises if libmlcc.so is missing: no fallback
    return a


def dev(x, dtype=torch.float64):
    return torch.as_tensor(np.ascontiguousarray(x), dtype=dtype).cuda()


def random_tables(rng, S, n):
    """a successor table made of S random permutations of n columns"""
    return np.stack([rng.permutation(n) for _ in range(S)]).astype(np.int32)


def assert_loops_equal(api, orc, nxt):
    col, end, lid, cnt = api.closed_loops(dev(nxt, torch.int32))
    ref = orc.closed_loops(nxt)
    assert np.array_equal(col.cpu().numpy(), ref["chain_col"])
    assert np.array_equal(end.cpu().numpy(), ref["chain_end"])
    assert np.array_equal(lid.cpu().numpy(), ref["loop_id"])
    assert int(cnt.item()) == ref["num_loops"]
    col2, end2, lid2, cnt2 = api.closed_loops(dev(nxt, torch.int32), want_chain_col=False)
    assert col2 is None and torch.equal(end2, end) and torch.equal(lid2, lid) and torch.equal(cnt2, cnt)
    return ref


# ---------------------------------------------------------------------------------------------
# closed loops
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("S,n", [(1, 1), (1, 7), (2, 1), (17, 95), (100, 256), (101, 257), (1000, 20), (37, 3000)])
def test_closed_loops_of_random_tables(api, orc, S, n):
    """Random permutations in every row: sizes below, at and above the 256-thread CTA and the sqrt(S) row blocks."""
    rng = np.random.default_rng(1000 * S + n)
    ref = assert_loops_equal(api, orc, random_tables(rng, S, n))
    assert ref["num_loops"] >= 1 and (ref["loop_id"] >= 0).all()


def test_closed_loops_long_cycle_and_identity(api, orc):
    """One cycle through all n chains (the most pointer-jumping rounds) and n fixed points."""
    n, S = 5000, 12
    nxt = np.tile(np.arange(n, dtype=np.int32), (S, 1))
    ref = assert_loops_equal(api, orc, nxt)
    assert ref["num_loops"] == n
    nxt[S - 1] = np.roll(np.arange(n), -1)
    ref = assert_loops_equal(api, orc, nxt)
    assert ref["num_loops"] == 1 and (ref["loop_id"] == 0).all()


def test_closed_loops_broken_and_non_bijective_tables(api, orc):
    """-1 entries (rows mlcc_link_rows could not link) and rows that are not bijections (two chains run into one
    column: a tail leading into a cycle).  Chains that are not on a cycle are labelled -1 on both sides."""
    rng = np.random.default_rng(3)
    S, n = 29, 300
    nxt = random_tables(rng, S, n)
    bad = nxt.copy()
    bad[11, rng.choice(n, 5, replace=False)] = -1
    bad[20, 7] = n + 3                                   # outside [0, n): treated like -1
    ref = assert_loops_equal(api, orc, bad)
    assert 5 <= (ref["chain_end"] == -1).sum() <= 6 and (ref["loop_id"] == -1).sum() >= 5
    rho = nxt.copy()
    rho[5, 10] = rho[5, 11]                              # columns 10 and 11 of row 5 both continue in the same column
    rho[17, 100:103] = rho[17, 200]
    ref = assert_loops_equal(api, orc, rho)
    assert (ref["loop_id"] == -1).any() and (ref["loop_id"] >= 0).any()
    every = np.full((4, 6), -1, np.int32)                # nothing links
    ref = assert_loops_equal(api, orc, every)
    assert ref["num_loops"] == 0


@pytest.mark.parametrize("name,num_phi", [("cfg1", 1000), ("cfg2", 800)])
def test_loops_of_the_critical_curves_end_to_end(api, orc, name, num_phi):
    """Each side runs its own whole chain: roots -> joining -> loops.  Column orders differ between the two, so
    what is unique is compared: the number of closed critical curves and the partition of the roots of row 0
    into them (GPU and oracle roots of row 0 paired by nearest neighbour)."""
    cfg = CONFIGS[name]
    xy, m, R = orc.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
    roots, iters, unconv, st = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi, cfg.tol,
                                                      cfg.max_iter)
    assert int(unconv.sum()) == 0
    nxt, bij = api.link_rows(roots)
    assert bool(bij.all())
    col, end, lid, cnt = api.closed_loops(nxt)
    o_roots, _, un = orc.critical_curves(xy, m, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter)
    assert un.sum() == 0
    o_nxt, o_bij = orc.link_rows(o_roots)
    assert o_bij.all()
    ref = orc.closed_loops(o_nxt)
    assert int(cnt.item()) == ref["num_loops"] and 1 <= ref["num_loops"] <= 2 * cfg.N
    from scipy.spatial import cKDTree
    g0 = roots[0].cpu().numpy()
    dist, to_orc = cKDTree(o_roots[0]).query(g0)                 # GPU column k of row 0 = oracle column to_orc[k]
    assert dist.max() < 1e-9 and len(set(to_orc.tolist())) == len(to_orc)
    g_lid = lid.cpu().numpy()
    g_sets = {frozenset(to_orc[g_lid == l].tolist()) for l in np.unique(g_lid)}
    o_sets = {frozenset(np.nonzero(ref["loop_id"] == l)[0].tolist()) for l in np.unique(ref["loop_id"])}
    assert g_sets == o_sets
    # the oracle's answer for the GPU's own table, exactly
    ref_g = orc.closed_loops(nxt.cpu().numpy())
    assert np.array_equal(col.cpu().numpy(), ref_g["chain_col"]) and np.array_equal(g_lid, ref_g["loop_id"])
    # chain order: every column is one continuous curve, also across the wrap to the next chain
    ordered = api.order_by_chain(roots, col)
    z = cplx(ordered.cpu().numpy())
    raw_jump = np.abs(np.diff(cplx(roots.cpu().numpy()), axis=0)).max()
    assert np.abs(np.diff(z, axis=0)).max() < 0.25 and raw_jump > 1.0     # raw columns jump between sub-chains
    assert np.abs(z[-1] - z[0][end.cpu().numpy()]).max() < 0.25


def test_order_by_chain_is_a_row_gather(api):
    rng = np.random.default_rng(9)
    S, n = 53, 777
    pts = rng.normal(size=(S, n, 2))
    col = random_tables(rng, S, n)
    col[3, 5] = -1
    col[8, 0] = n
    out = api.order_by_chain(dev(pts), dev(col, torch.int32)).cpu().numpy()
    safe = np.clip(col, 0, n - 1)
    want = np.take_along_axis(pts, safe[:, :, None], axis=1)
    ok = (col >= 0) & (col < n)
    assert np.array_equal(out[ok], want[ok]) and np.isnan(out[~ok]).all() and (~ok).sum() == 2
    empty = api.order_by_chain(torch.empty((0, 4, 2), dtype=torch.float64, device="cuda"),
                               torch.empty((0, 4), dtype=torch.int32, device="cuda"))
    assert empty.shape == (0, 4, 2)


def test_closed_loops_full_size_cfg4_table(api, orc):
    """The size of cfg4's table (10^4 rows x 2*10^4 columns, 800 MB): near-identity permutations with a few swaps per
    row as between sub-chains, checked by properties that hold at any size and against the oracle on the table."""
    S, n = 10_000, 20_000
    g = torch.Generator(device="cpu").manual_seed(5)
    nxt = torch.arange(n, dtype=torch.int32).repeat(S, 1)
    rows = torch.randint(0, S, (4000,), generator=g)
    a = torch.randint(0, n, (4000,), generator=g)
    b = torch.randint(0, n, (4000,), generator=g)
    for r, i, j in zip(rows.tolist(), a.tolist(), b.tolist()):   # swap two entries of a row: still a permutation
        t = int(nxt[r, i]); nxt[r, i] = nxt[r, j]; nxt[r, j] = t
    col, end, lid, cnt = api.closed_loops(nxt.cuda())
    torch.cuda.synchronize()
    ref = orc.closed_loops(nxt.numpy(), want_chain_col=False)
    assert np.array_equal(end.cpu().numpy(), ref["chain_end"])
    assert np.array_equal(lid.cpu().numpy(), ref["loop_id"]) and int(cnt.item()) == ref["num_loops"]
    c = col.cpu()
    assert torch.equal(c[0], torch.arange(n, dtype=torch.int32))
    s = torch.randint(0, S - 1, (64,), generator=g)
    for r in s.tolist():                                          # the recurrence, on sampled rows
        assert torch.equal(c[r + 1], nxt[r][c[r].long()])
    assert torch.equal(end.cpu(), nxt[S - 1][c[S - 1].long()])
    assert torch.equal(torch.sort(c[S // 2]).values, torch.arange(n, dtype=torch.int32))   # a permutation


# ---------------------------------------------------------------------------------------------
# distance maps
# ---------------------------------------------------------------------------------------------
def crossing_map_of(orc, name, num_phi, n_pix):
    cfg = CONFIGS[name]
    xy, m, R = orc.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
    roots, _, un = orc.critical_curves(xy, m, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter)
    assert un.sum() == 0
    caus = orc.caustics(xy, m, cfg.kappa_s, cfg.gamma, roots)
    nxt, bij = orc.link_rows(roots)
    assert bij.all()
    z = cplx(caus).ravel()
    c, half = (z.real.min() + z.real.max()) / 2 + 1j * (z.imag.min() + z.imag.max()) / 2, 0.3 * np.ptp(z.real)
    pixel = 2 * half / n_pix
    return orc.crossing_map(caus, nxt, c.real - half, c.imag - half, pixel, n_pix, n_pix), pixel


@pytest.mark.parametrize("nx,ny", [(1, 1), (1, 40), (40, 1), (37, 23), (64, 64), (257, 100), (90, 300)])
def test_distance_map_against_oracle(api, orc, nx, ny):
    rng = np.random.default_rng(nx * 1000 + ny)
    m = blob_map(rng, nx, ny) if min(nx, ny) > 1 else rng.integers(0, 2, size=(ny, nx)).astype(np.int32)
    ref, ref2 = orc.distance_map(m, 0.37)
    got, got2 = api.distance_map(dev(m, torch.int32), 0.37, want_d2=True)
    assert np.array_equal(got2.cpu().numpy(), ref2)
    assert np.allclose(got.cpu().numpy(), ref, rtol=1e-15, atol=0)
    assert torch.equal(api.distance_map(dev(m, torch.int32), 0.37), got)


def test_distance_map_without_caustics_is_infinite(api, orc):
    flat = np.full((9, 14), 2, np.int32)
    got, got2 = api.distance_map(dev(flat, torch.int32), 1.0, want_d2=True)
    assert bool(torch.isinf(got).all()) and bool((got2 == -1).all())
    one = flat.copy()
    one[4, 6] = 3                                      # the pixel and its four neighbours become caustic pixels
    ref, ref2 = orc.distance_map(one, 1.0)
    got, got2 = api.distance_map(dev(one, torch.int32), 1.0, want_d2=True)
    assert np.array_equal(got2.cpu().numpy(), ref2) and (ref2 == 0).sum() == 5


def test_distance_maps_of_a_caustic_network(api, orc):
    """The oracle's own crossing map of cfg1 (oracle roots -> caustics -> joining -> winding numbers) as the input
    of both sides, for both maps."""
    cmap, pixel = crossing_map_of(orc, "cfg1", 720, 96)
    assert cmap.max() >= 2
    ref, ref2 = orc.distance_map(cmap, pixel)
    got, got2 = api.distance_map(dev(cmap, torch.int32), pixel, want_d2=True)
    assert np.array_equal(got2.cpu().numpy(), ref2) and np.allclose(got.cpu().numpy(), ref, rtol=1e-15, atol=0)
    for ux, uy in [(0, 1), (1, 0), (-3, 2), (5, -7)]:
        ref = orc.directional_distance_map(cmap, pixel, ux, uy)
        got = api.directional_distance_map(dev(cmap, torch.int32), pixel, ux, uy).cpu().numpy()
        assert np.array_equal(np.sign(got), np.sign(ref)) and np.allclose(got, ref, rtol=1e-15, atol=0)
        # along the direction of motion a caustic is never nearer than the nearest one in any direction;
        # a caustic pixel of the transform lies at most one pixel diagonal behind the border the ray stops at
        hit = ref > 0
        d_any = orc.distance_map(cmap, pixel)[0]
        assert (ref[hit] + np.sqrt(2.0) * pixel >= d_any[hit]).all()


@pytest.mark.parametrize("ux,uy", [(1, 0), (-1, 0), (0, 1), (0, -1), (1, 1), (-1, 1), (2, 1), (-3, -5), (7, -2),
                                   (1024, 1), (1, -1000), (1 << 20, (1 << 20) - 1)])
def test_directional_distance_against_oracle(api, orc, ux, uy):
    rng = np.random.default_rng(abs(ux) * 7 + abs(uy))
    for nx, ny in [(33, 47), (64, 20), (1, 9), (300, 2)]:
        m = blob_map(rng, nx, ny, blobs=4) if min(nx, ny) > 2 else rng.integers(0, 3, size=(ny, nx)).astype(np.int32)
        ref = orc.directional_distance_map(m, 0.5, ux, uy)
        got = api.directional_distance_map(dev(m, torch.int32), 0.5, ux, uy).cpu().numpy()
        assert np.array_equal(np.sign(got), np.sign(ref))
        assert np.allclose(got, ref, rtol=1e-15, atol=0), np.abs(got - ref).max()


def test_distance_maps_full_size(api, orc):
    """2048 x 1536 pixels (the oracle's brute force is O(P^2)): the transform against scipy's exact Euclidean distance
    transform of the same mask -- the routine the oracle is pinned to on the CPU -- and the moving-source map by the
    property that one pixel further along an axis inside the same region the caustic is exactly one pixel nearer."""
    ndi = pytest.importorskip("scipy.ndimage")
    from test_oracle_loops_distance import edge_mask
    rng = np.random.default_rng(77)
    nx, ny, pixel = 2048, 1536, 0.03
    m = blob_map(rng, nx, ny, blobs=40)
    got, got2 = api.distance_map(dev(m, torch.int32), pixel, want_d2=True)
    e = edge_mask(m)
    ref = ndi.distance_transform_edt(~e)
    assert np.array_equal(got2.cpu().numpy(), np.rint(ref ** 2).astype(np.int64))
    assert np.allclose(got.cpu().numpy(), pixel * ref, rtol=1e-15, atol=0)
    # sampled pixels one by one with the oracle: a window around the pixel that holds its nearest caustic pixel
    # (the nearest caustic pixel and the neighbour that makes it one lie inside the window, and every caustic pixel
    # of the window is one of the map)
    g2 = got2.cpu().numpy()
    ys, xs = np.nonzero((g2 > 0) & (g2 <= 20 ** 2))
    for q in rng.choice(len(ys), size=12, replace=False):
        x, y = int(xs[q]), int(ys[q])
        r = int(np.ceil(np.sqrt(g2[y, x]))) + 2
        x0, x1, y0, y1 = max(x - r, 0), min(x + r + 1, nx), max(y - r, 0), min(y + r + 1, ny)
        d_sub, d2_sub = orc.distance_map(m[y0:y1, x0:x1], pixel)
        assert d2_sub[y - y0, x - x0] == g2[y, x]
    d = api.directional_distance_map(dev(m, torch.int32), pixel, 1, 0).cpu().numpy()
    same = m[:, 1:] == m[:, :-1]
    assert np.allclose((np.abs(d[:, :-1]) - np.abs(d[:, 1:]))[same], pixel, rtol=0, atol=1e-12)
    assert np.array_equal(np.sign(d[:, :-1])[same], np.sign(d[:, 1:])[same])
    assert np.allclose(d[:, :-1][~same], 0.5 * pixel, rtol=1e-15)
    assert np.allclose(d[:, -1], -0.5 * pixel, rtol=1e-15)
    d = api.directional_distance_map(dev(m, torch.int32), pixel, 0, -1).cpu().numpy()
    same = m[1:, :] == m[:-1, :]
    assert np.allclose((np.abs(d[1:, :]) - np.abs(d[:-1, :]))[same], pixel, rtol=0, atol=1e-12)
    assert np.allclose(d[0, :], -0.5 * pixel, rtol=1e-15)


@pytest.mark.parametrize("num_bins,num_counts", [(16, 5), (1, 1), (4096, 2), (5000, 4)])
def test_distance_histogram_against_oracle(api, orc, num_bins, num_counts):
    """Small tables (counted in shared memory) and one beyond 8192 entries (global atomics); negative, infinite and NaN
    distances and out-of-range counts on both sides.  Integer counts: exact."""
    rng = np.random.default_rng(num_bins + num_counts)
    shape = (301, 517)
    d = rng.uniform(0, 6, size=shape)
    d[rng.random(shape) < 0.1] *= -1
    d[rng.random(shape) < 0.01] = np.inf
    d[rng.random(shape) < 0.01] = np.nan
    d[0, :7] = 0.5 * np.arange(7)                        # values on bin edges
    cm = rng.integers(-2, 8, size=shape).astype(np.int32)
    bw = 5.0 / num_bins if num_bins > 1 else 0.5
    for cmap in (cm, None):
        ref, ref_left = orc.distance_histogram(d, cmap, bw, num_bins, num_counts)
        got, left = api.distance_histogram(dev(d), None if cmap is None else dev(cmap, torch.int32), bw, num_bins,
                                           num_counts)
        assert np.array_equal(got.cpu().numpy(), ref) and int(left.item()) == ref_left
        assert ref.sum() + ref_left == d.size
    empty = api.distance_histogram(torch.empty((0, 5), dtype=torch.float64, device="cuda"), None, 0.5, 4)
    assert int(empty[0].sum()) == 0 and int(empty[1].item()) == 0


def test_distance_statistics_of_a_caustic_network(api, orc):
    """Fig. 6 / Fig. 7 on the oracle's crossing map of cfg1: histogram of the moving-source distance per direction,
    and of the distance between the caustics before and behind the source split by the crossing count."""
    cmap, pixel = crossing_map_of(orc, "cfg1", 720, 96)
    g_map = dev(cmap, torch.int32)
    for ux, uy in [(1, 0), (0, 1), (2, 3)]:
        fwd = api.directional_distance_map(g_map, pixel, ux, uy)
        bwd = api.directional_distance_map(g_map, pixel, -ux, -uy)
        o_fwd = orc.directional_distance_map(cmap, pixel, ux, uy)
        o_bwd = orc.directional_distance_map(cmap, pixel, -ux, -uy)
        ref, ref_left = orc.distance_histogram(o_fwd, None, 2 * pixel, 24)
        got, left = api.distance_histogram(fwd, None, 2 * pixel, 24)
        assert np.array_equal(got.cpu().numpy(), ref) and int(left.item()) == ref_left and ref.sum() > 1000
        both = torch.where((fwd > 0) & (bwd > 0), fwd + bwd, torch.full_like(fwd, -1.0))
        o_both = np.where((o_fwd > 0) & (o_bwd > 0), o_fwd + o_bwd, -1.0)
        ref, ref_left = orc.distance_histogram(o_both, cmap, 2 * pixel, 24, int(cmap.max()) + 1)
        got, left = api.distance_histogram(both, g_map, 2 * pixel, 24, int(cmap.max()) + 1)
        assert np.array_equal(got.cpu().numpy(), ref) and int(left.item()) == ref_left
        # every pixel inside a caustic (count >= 1) whose chord ends on caustics at both ends is in the table or left out
        inside = (cmap >= 1) & (o_both > 0)
        assert ref[1:].sum() == (inside & (np.floor(o_both / (2 * pixel)) < 24)).sum() > 0


def test_argument_checks(api):
    cm = torch.zeros((4, 4), dtype=torch.int32, device="cuda")
    with pytest.raises(api.MlccError) as e:
        api.directional_distance_map(cm, 1.0, 0, 0)
    assert e.value.status == api.MLCC_ERR_INVALID_ARG
    with pytest.raises(api.MlccError):
        api.directional_distance_map(cm, 1.0, (1 << 20) + 1, 0)
    with pytest.raises(api.MlccError):
        api.distance_map(cm, 0.0)
    with pytest.raises(TypeError):
        api.distance_map(cm.cpu(), 1.0)
    with pytest.raises(TypeError):
        api.closed_loops(torch.zeros((3, 3), dtype=torch.int64, device="cuda"))
