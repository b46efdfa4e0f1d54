"""GPU parity tests: the CUDA path (through the C-ABI binding) against the CPU oracle on the same
seeded inputs.  All inputs are generated on the CPU by the oracle's generator and uploaded; no oracle
input or expected value comes from the CUDA path.

Tolerances (BASELINE.json north_star): root sets per phase after nearest-neighbour matching
max |dz| <= 1e-10 (1 + |z|); caustic points within 1e-9; integer outputs exact.
"""
import numpy as np
import pytest

from paper_2506_02121_b200.configs import CONFIGS
from test_oracle_pins import check_row_invariants, c_phi, cplx

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

ROOT_TOL = 1e-10
CAUSTIC_TOL = 1e-9


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2506_02121_b200 import api as a
    a.lib()  # raises if libmlcc.so is missing: no fallback
    return a


def dev(x, dtype=torch.float64):
    return torch.as_tensor(np.ascontiguousarray(x), dtype=dtype).cuda()


def field(orc, cfg, N=None):
    return orc.star_field(cfg.seed, N or cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)


def assert_rows_match(orc, gpu_rows, ref_rows, tol=ROOT_TOL):
    """gpu_rows, ref_rows: [S, n, 2] numpy.  Oracle brute-force matching, b = reference."""
    err, bij = orc.match_root_sets(gpu_rows, ref_rows, tol)
    assert bij.all(), (np.where(bij == 0)[0][:10], err.max())
    return err.max()


def assert_caustics_match(g_roots, g_caus, ref_roots, ref_caus, tol=CAUSTIC_TOL):
    """One row each: pair GPU roots with oracle roots (KD-tree), compare their caustic points."""
    from scipy.spatial import cKDTree
    dist, perm = cKDTree(ref_roots).query(g_roots)
    assert len(set(perm.tolist())) == len(perm)
    assert np.abs(cplx(g_caus) - cplx(ref_caus)[perm]).max() <= tol


# ---------------------------------------------------------------------------------------------
# a0 star field
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["cfg1", "cfg3", "cfg4", "cfg5"])
def test_star_field_matches_oracle_generator(api, orc, name):
    cfg = CONFIGS[name]
    xy, m, R = api.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
    oxy, om, oR = field(orc, cfg)
    assert R == oR
    assert np.array_equal(xy.cpu().numpy(), oxy)            # positions: bit-exact
    assert np.abs(m.cpu().numpy() / om - 1).max() < 1e-14   # masses: pow() may differ by a few ulp
    assert abs(float(m.sum()) - cfg.N) < 1e-9 * cfg.N


@pytest.mark.parametrize("N,kstar,aspect,model", [(1, 0.4, 1.0, 0), (600, 0.4, 2.0, 1), (10000, 0.2, 0.5, 2),
                                                  (50001, 0.6, 1.3, 0)])
def test_rectangular_star_field_matches_oracle_generator(api, orc, N, kstar, aspect, model):
    """mlcc_star_field_rect (Section 4.2's field): corner and positions bit-exact, masses to a few ulp."""
    xy, m, c1, c2 = api.star_field_rect(7, N, kstar, aspect, model)
    oxy, om, oc1, oc2 = orc.star_field_rect(7, N, kstar, aspect, model)
    assert (c1, c2) == (oc1, oc2)
    assert np.array_equal(xy.cpu().numpy(), oxy)
    assert np.abs(m.cpu().numpy() / om - 1).max() < 1e-14
    with pytest.raises(api.MlccError):
        api.star_field_rect(7, N, kstar, -1.0, model)


def test_star_field_seed_and_defaults(api, orc):
    a = api.star_field(5, 1000, 0.3, 2)
    b = api.star_field(5, 1000, 0.3, 2, (0.01, 0.08, 0.5, 1.5, 0.3, 1.3, 2.3))
    c = api.star_field(6, 1000, 0.3, 2)
    assert torch.equal(a[0], b[0]) and torch.equal(a[1], b[1])
    assert not torch.equal(a[0], c[0])
    oxy, om, _ = orc.star_field(5, 1000, 0.3, 1, (0.1, 2.0, 1.0))   # alpha = 1 branch
    gxy, gm, _ = api.star_field(5, 1000, 0.3, 1, (0.1, 2.0, 1.0))
    assert np.array_equal(gxy.cpu().numpy(), oxy) and np.abs(gm.cpu().numpy() / om - 1).max() < 1e-14


# ---------------------------------------------------------------------------------------------
# a1-a6 critical curves, a7 caustics: full grids where the oracle finishes in seconds
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("regime", [1, 2])
@pytest.mark.parametrize("name", ["cfg1", "cfg2"])
def test_curves_and_caustics_full_grid(api, orc, name, regime):
    """Full grids of cfg1 / cfg2 against the oracle, in both kernel regimes (1 = tiled launches, 2 = one CTA per
    sub-chain: mlcc_options.regime)."""
    cfg = CONFIGS[name]
    xy, m, R = field(orc, cfg)
    ref, it_ref, un_ref = orc.critical_curves(xy, m, cfg.kappa_s, cfg.gamma, cfg.num_phi, cfg.tol, cfg.max_iter)
    assert un_ref.sum() == 0
    roots, iters, unconv, stats = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, cfg.num_phi,
                                                         cfg.tol, cfg.max_iter, opt=api.options(regime=regime))
    assert stats.regime == regime
    assert int(unconv.sum()) == 0 and stats.unconverged_rows == 0 and stats.degenerate_roots == 0
    assert int(iters.min()) >= 1 and int(iters.max()) <= cfg.max_iter
    assert stats.root_iterations >= cfg.num_phi * 2 * cfg.N
    again, _, _, _ = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, cfg.num_phi, cfg.tol, cfg.max_iter,
                                            opt=api.options(regime=regime))
    assert torch.equal(again, roots)                      # fixed summation order: two runs give the same bits
    certify_every_row(api, dev(xy), dev(m), cfg, roots)
    g = roots.cpu().numpy()
    assert_rows_match(orc, g, ref)
    # caustics: GPU roots -> GPU caustics, oracle roots -> oracle caustics, compared through the matching
    w_gpu = api.caustics(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, roots).cpu().numpy()
    w_ref = orc.caustics(xy, m, cfg.kappa_s, cfg.gamma, ref)
    for j in range(0, cfg.num_phi, max(1, cfg.num_phi // 200)):
        assert_caustics_match(g[j], w_gpu[j], ref[j], w_ref[j])
    # the same points through both caustic maps, element by element
    w_same = api.caustics(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, dev(ref)).cpu().numpy()
    assert np.abs(w_same - w_ref).max() <= 1e-12 * (1 + np.abs(w_ref).max())
    # default-options entry point on the default stream
    r2 = api.critical_curves(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, cfg.num_phi, cfg.tol, cfg.max_iter)
    if regime == 2:                                       # the regime AUTO picks for these fields
        assert torch.equal(r2, roots)
    else:
        assert_rows_match(orc, r2.cpu().numpy(), ref)


# ---------------------------------------------------------------------------------------------
# full-size runs of the larger configs in the launch configuration bench.py times (default options):
# oracle on sampled rows; invariants that hold at any size on all / many rows
# ---------------------------------------------------------------------------------------------
def vieta_all_rows(roots, xy, m, kappa_s, gamma, num_phi):
    """sum z_k = 2 sum z_i and sum z_k^2 = 2 sum z_i^2 + 2 sum m / c(phi) on every row (torch on the device)."""
    z = torch.view_as_complex(roots)
    zs = torch.view_as_complex(dev(xy))
    phi = 2 * np.pi * torch.arange(num_phi, device="cuda", dtype=torch.float64) / num_phi
    c = (1 - kappa_s) * torch.exp(-1j * phi) - gamma
    s1 = z.sum(dim=1)
    s2 = (z * z).sum(dim=1)
    scale1 = z.abs().sum(dim=1)
    scale2 = (z.abs() ** 2).sum(dim=1)
    e1 = (s1 - 2 * zs.sum()).abs() / scale1
    e2 = (s2 - (2 * (zs * zs).sum() + 2 * float(m.sum()) / c)).abs() / scale2
    return float(e1.max()), float(e2.max())


def certify_every_row(api, xy_d, m_d, cfg, roots, phi_off=0, phi_total=0):
    """mlcc_detj_residuals on EVERY row (BASELINE.json north_star: "|det J| <= 1e-10 at every root", with the scale-aware
    bound of SURVEY.md 0.2): max_k |1/mu_k| / bound_k <= 1 and max_k |F|/|F'| far inside the parity tolerance, so a
    root that stopped 1e-9 from its place cannot pass (Vieta's sums would not see it)."""
    rn, rd, _ = api.detj_residuals(xy_d, m_d, cfg.kappa_s, cfg.gamma, roots, phi_off, phi_total)
    assert float(rd.max()) <= 1.0, (int(rd.argmax()), float(rd.max()))
    assert float(rn.max()) < 1e-11, (int(rn.argmax()), float(rn.max()))
    return rn, rd


def rows_beside_the_centres(api, cfg, which, halfwidth=2):
    """Rows centre-halfwidth .. centre+halfwidth of the listed sub-chains of the library's default plan: the rows whose
    predictor stencil is shortened (the first continued rows of a chain)."""
    first, centre, end = api.plan_subchains(cfg.N, cfg.num_phi, 0)
    out = []
    for c in which:
        c = c % len(centre)
        out.append([int(r) for r in range(int(centre[c]) - halfwidth, int(centre[c]) + halfwidth + 1)
                    if first[c] <= r < end[c]])
    return out, len(centre)


@pytest.mark.parametrize("name,sample_rows,centres,halfwidth", [("cfg3", [0, 1, 1250, 2499, 2500, 4999], [0, 17], 2),
                                                                 ("cfg4", [0, 4999, 9999], [0, 5], 2),
                                                                 ("cfg5", [], [1], 1)])
def test_full_size_sampled_rows_and_invariants(api, orc, name, sample_rows, centres, halfwidth):
    cfg = CONFIGS[name]
    xy, m, R = field(orc, cfg)
    roots, iters, unconv, stats = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, cfg.num_phi,
                                                         cfg.tol, cfg.max_iter)
    torch.cuda.synchronize()
    assert int(unconv.sum()) == 0 and stats.degenerate_roots == 0
    assert int(iters.min()) >= 1
    # properties that hold at any size, every row: Vieta sums (complete, no duplicated root), det J and Newton residual
    e1, e2 = vieta_all_rows(roots, xy, m, cfg.kappa_s, cfg.gamma, cfg.num_phi)
    assert e1 < 1e-12 and e2 < 1e-12, (e1, e2)
    certify_every_row(api, dev(xy), dev(m), cfg, roots)
    # sampled rows against the oracle (each row cold-started by the oracle on its own)
    for j in sample_rows:
        ref, _, un = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, cfg.num_phi, [j], cfg.tol, cfg.max_iter)
        assert un.sum() == 0
        g = roots[j:j + 1].cpu().numpy()
        assert_rows_match(orc, g, ref)
        # caustic points of that row
        w_gpu = api.caustics(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, roots[j:j + 1].contiguous()).cpu().numpy()
        w_ref = orc.caustics(xy, m, cfg.kappa_s, cfg.gamma, ref)
        assert_caustics_match(g[0], w_gpu[0], ref[0], w_ref[0])
    # the rows beside sub-chain centres (cold row, then the rows seeded with a shortened predictor stencil): the oracle
    # cold-starts the first of them and continues through the rest
    groups, n_sub = rows_beside_the_centres(api, cfg, centres, halfwidth)
    assert n_sub == stats.subchains
    oracle_row = {}
    for rows in groups:
        ref, _, un = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, cfg.num_phi, rows, cfg.tol, cfg.max_iter)
        assert un.sum() == 0
        g = roots[rows[0]:rows[-1] + 1].cpu().numpy()
        assert_rows_match(orc, g, ref)
        oracle_row[rows[0]] = ref[0]
    # certificates on more rows than the oracle can solve: long-double residuals, det J, distinctness; and the kernel's
    # worst long-double residual of a row is held to twice that of the oracle's own fp64 solve of the same row
    rng = np.random.default_rng(1)
    extra = [groups[0][0]] if groups else []
    for j in list(rng.choice(cfg.num_phi, size=4, replace=False)) + extra:
        res = check_row_invariants(orc, xy, m, cfg.kappa_s, cfg.gamma, int(j), cfg.num_phi,
                                   cplx(roots[int(j)].cpu().numpy()))
        if int(j) in extra:
            worst_gpu = res["newton"].max()
            res_o = orc.residuals(xy, m, cfg.kappa_s, cfg.gamma, int(j), cfg.num_phi, oracle_row[int(j)])   # the oracle's fp64 solve
            assert worst_gpu <= 2 * res_o["newton"].max() + 1e-13, (worst_gpu, res_o["newton"].max())


@pytest.mark.parametrize("name,rows", [("cfg1", [0, 499, 500]), ("cfg2", [0, 7, 2000]), ("cfg3", [1250]), ("cfg4", [0])])
def test_detj_residuals_against_oracle(api, orc, name, rows):
    """mlcc_detj_residuals element by element against the oracle's long-double F, F', 1/mu, |F|/|F'| (orc_residuals_ld):
    at converged roots (where F is a rounding-level residue of terms of size sum |m/(z-z_i)^2|) and at displaced
    points (where F is O(1) and the comparison is relative)."""
    cfg = CONFIGS[name]
    xy, m, R = field(orc, cfg)
    zs = xy[:, 0] + 1j * xy[:, 1]
    ref, _, un = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, cfg.num_phi, rows[:1], cfg.tol, cfg.max_iter)
    assert un.sum() == 0
    rng = np.random.default_rng(5)
    n = min(2 * cfg.N, 4000)                                          # (n is free: a part of the row is enough at N = 10^4)
    pts = np.empty((len(rows), n, 2))
    pts[0] = ref[0][-n:]                                              # converged roots (phase of rows[0])
    for q in range(1, len(rows)):                                     # displaced points, other phases
        pts[q] = ref[0][-n:] + rng.normal(scale=0.05, size=(n, 2))
    xy_d, m_d = dev(xy), dev(m)
    for q, j in enumerate(rows):
        rn, rd, res = api.detj_residuals(xy_d, m_d, cfg.kappa_s, cfg.gamma, dev(pts[q:q + 1]), j, cfg.num_phi,
                                         want_points=True)
        res = res.cpu().numpy()[0]
        o = orc.residuals(xy, m, cfg.kappa_s, cfg.gamma, j, cfg.num_phi, pts[q])
        z = pts[q, :, 0] + 1j * pts[q, :, 1]
        d = np.abs(z[:, None] - zs[None, :])
        t2 = (m[None, :] / d ** 2).sum(axis=1) + abs(cfg.gamma) + (1 - cfg.kappa_s)      # size of the terms of F
        t3 = 2 * (m[None, :] / d ** 3).sum(axis=1)                                         # ... of F'
        F, Fp = res[:, 0] + 1j * res[:, 1], res[:, 2] + 1j * res[:, 3]
        assert (np.abs(F - o["F"]) <= 1e-12 * t2).all()
        assert (np.abs(Fp - o["Fp"]) <= 1e-12 * t3).all()
        assert (np.abs(res[:, 4] - o["inv_mu"]) <= 1e-12 * t2 ** 2).all()
        assert (np.abs(res[:, 5] - o["newton"]) <= 1e-12 * t2 / np.abs(o["Fp"]) + 1e-12 * o["newton"] * t3 / np.abs(o["Fp"])).all()
        # the row outputs are the maxima of the point outputs
        bound = 1e-10 + 4 * (1 - cfg.kappa_s) * np.abs(Fp) * 2.0 ** -52 * (1 + np.abs(z))
        assert float(rn[0]) == res[:, 5].max()
        assert abs(float(rd[0]) - (np.abs(res[:, 4]) / bound).max()) <= 1e-12 * float(rd[0])
        if q == 0:
            assert float(rd[0]) <= 1.0 and float(rn[0]) < 1e-11       # the oracle's own converged row is certified
        else:
            assert float(rd[0]) > 1.0                                 # displaced points are not
    # several rows in one call = the rows one by one; a wrong phase offset is seen; a point on a star gives +inf
    rn_all, rd_all, _ = api.detj_residuals(xy_d, m_d, cfg.kappa_s, cfg.gamma, dev(np.repeat(pts[:1], 3, axis=0)), rows[0],
                                           cfg.num_phi)
    # det J = 0 on the critical curve whatever phi is: only the Newton residual of F sees the phase (rows[0]+1, +2)
    assert float(rd_all.max()) <= 1.0 and float(rn_all[0]) < 1e-11 and float(rn_all[1]) > 1e-7 and float(rn_all[2]) > float(rn_all[1])
    bad = pts[:1].copy()
    bad[0, 3] = xy[0]
    rn_b, rd_b, _ = api.detj_residuals(xy_d, m_d, cfg.kappa_s, cfg.gamma, dev(bad), rows[0], cfg.num_phi)
    assert np.isinf(float(rn_b[0])) or np.isinf(float(rd_b[0]))
    empty = api.detj_residuals(xy_d, m_d, cfg.kappa_s, cfg.gamma, torch.empty((0, n, 2), dtype=torch.float64, device="cuda"))
    assert empty[0].shape == (0,)


@pytest.mark.parametrize("name,num_phi", [("cfg1", 1000), ("cfg2", 777), ("cfg3", 64)])
def test_vieta_residuals_against_oracle(api, orc, name, num_phi):
    """mlcc_vieta_residuals (the validator's invariant half) on GPU root sets: tiny on every row, equal to the oracle's
    long-double evaluation within rounding; a duplicated root and a wrong phase offset are reported by both alike."""
    cfg = CONFIGS[name]
    xy, m, R = field(orc, cfg)
    roots, _, unconv, _ = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter)
    assert int(unconv.sum()) == 0
    e1, e2 = api.vieta_residuals(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, roots)
    o1, o2 = orc.vieta_residuals(xy, m, cfg.kappa_s, cfg.gamma, roots.cpu().numpy())
    assert float(e1.max()) < 1e-12 and float(e2.max()) < 1e-12 and o1.max() < 1e-12 and o2.max() < 1e-12
    assert np.abs(e1.cpu().numpy() - o1).max() < 1e-14 and np.abs(e2.cpu().numpy() - o2).max() < 1e-14
    bad = roots.clone()
    bad[5, 3] = bad[5, 4]                                  # row 5: one root twice, one missing
    bad[9, 0, 0] += 1e-6                                    # row 9: one root misplaced by 1e-6
    b1, b2 = api.vieta_residuals(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, bad)
    p1, p2 = orc.vieta_residuals(xy, m, cfg.kappa_s, cfg.gamma, bad.cpu().numpy())
    assert np.allclose(b1.cpu().numpy()[[5, 9]], p1[[5, 9]], rtol=1e-6) and np.allclose(b2.cpu().numpy()[[5, 9]], p2[[5, 9]], rtol=1e-6)
    assert float(b1[5]) > 1e-6 and float(b1[9]) > 1e-6 / float(roots[9].norm(dim=1).sum()) * 0.99
    ok = np.ones(num_phi, bool)
    ok[[5, 9]] = False
    assert float(b1.cpu().numpy()[ok].max()) < 1e-12
    # rows of a larger grid (multi-GPU sharding, mlcc_options.phi_index_offset / _total)
    part, _, _, _ = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, 16, cfg.tol, cfg.max_iter,
                                           opt=api.options(phi_index_offset=40, phi_index_total=num_phi))
    s1, s2 = api.vieta_residuals(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, part, 40, num_phi)
    q1, q2 = orc.vieta_residuals(xy, m, cfg.kappa_s, cfg.gamma, part.cpu().numpy(), 40, num_phi)
    assert float(s2.max()) < 1e-12 and q2.max() < 1e-12
    w1, w2 = api.vieta_residuals(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, part, 0, num_phi)       # wrong offset
    assert float(w2.min()) > 1e-9 and float(w1.max()) < 1e-12                                    # only the second sum has phi
    empty = api.vieta_residuals(dev(xy), dev(m), cfg.kappa_s, cfg.gamma,
                                torch.empty((0, 2 * cfg.N, 2), dtype=torch.float64, device="cuda"))
    assert empty[0].shape == (0,)


def test_bench_configuration_full_size_cfg4(api, orc):
    """The call bench.py times, as it times it: mlcc_star_field + the FUSED mlcc_curves_and_caustics with default
    options on cfg4 at its full size (10^4 phases x 2*10^4 roots) + mlcc_match_root_sets.  Sampled rows (roots and
    their fused caustic points) against the oracle, Vieta sums and the device validator on every row, and a second
    run that must give the same bits."""
    cfg = CONFIGS["cfg4"]
    xy, m, R = api.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
    oxy, om, oR = field(orc, cfg)
    assert R == oR and np.array_equal(xy.cpu().numpy(), oxy)
    xy_o, m_o = dev(oxy), dev(om)                    # both sides solve the oracle generator's field
    roots, caus, iters, unconv, st = api.curves_and_caustics(xy_o, m_o, cfg.kappa_s, cfg.gamma, cfg.num_phi, cfg.tol,
                                                             cfg.max_iter, want_diagnostics=False)
    assert st.unconverged_rows == 0 and st.degenerate_roots == 0 and st.subchains >= 2
    e1, e2 = vieta_all_rows(roots, oxy, om, cfg.kappa_s, cfg.gamma, cfg.num_phi)
    assert e1 < 1e-12 and e2 < 1e-12, (e1, e2)
    for j in (17, 5000, 7321, 9999):
        ref, _, un = orc.critical_curve_rows(oxy, om, cfg.kappa_s, cfg.gamma, cfg.num_phi, [j], cfg.tol, cfg.max_iter)
        assert un.sum() == 0
        g = roots[j:j + 1].cpu().numpy()
        assert_rows_match(orc, g, ref)
        w_ref = orc.caustics(oxy, om, cfg.kappa_s, cfg.gamma, ref)
        assert_caustics_match(g[0], caus[j].cpu().numpy(), ref[0], w_ref[0])
    g1, g2 = api.vieta_residuals(xy_o, m_o, cfg.kappa_s, cfg.gamma, roots)       # the library's own certificates
    assert float(g1.max()) < 1e-12 and float(g2.max()) < 1e-12
    certify_every_row(api, xy_o, m_o, cfg, roots)
    again, caus2, _, _, _ = api.curves_and_caustics(xy_o, m_o, cfg.kappa_s, cfg.gamma, cfg.num_phi, cfg.tol,
                                                    cfg.max_iter, want_diagnostics=False)
    err, bij = api.match_root_sets(again, roots, 1e-10)
    assert bool(bij.all()) and float(err.max()) == 0.0
    assert torch.equal(again, roots) and torch.equal(caus2, caus)


# ---------------------------------------------------------------------------------------------
# the chain regime (one CTA per sub-chain, chain.cu): sizes that exercise every pass shape and edge
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,num_phi,nsub", [(1, 1, 0), (1, 7, 0), (2, 33, 2), (3, 64, 0), (17, 101, 5), (64, 40, 0),
                                            (129, 96, 3), (300, 50, 0), (640, 24, 0), (1200, 12, 2)])
def test_chain_regime_sizes_and_edges(api, orc, N, num_phi, nsub):
    """Fields from one star (two roots, fewer roots than lanes: T-lane passes) to the largest that fits shared memory
    (N = 1200), grids that do not divide into the sub-chains, one-row sub-chains: root sets and fused caustic points
    against the oracle, diagnostics, and the tiled regime on the same input."""
    cfg = CONFIGS["cfg2"]
    xy, m, R = orc.star_field(11, N, cfg.kappa_star, 1, (0.08, 1.0, 2.35))
    if N == 1:
        xy = xy + np.array([[0.37, -0.21]])            # keep the single star (and its seeds) off the real axis
    dxy, dm = dev(xy), dev(m)
    opt = api.options(regime=2, num_subchains=nsub)
    roots, caus, iters, unconv, st = api.curves_and_caustics(dxy, dm, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter,
                                                             opt=opt)
    assert st.regime == 2 and st.kernel_launches == 2 and st.unconverged_rows == 0 and st.degenerate_roots == 0
    assert int(unconv.sum()) == 0 and int(iters.min()) >= 1
    assert st.root_iterations >= num_phi * 2 * N and st.star_pairs == st.root_iterations * N
    if N <= 300:
        ref, _, un = orc.critical_curves(xy, m, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter)
    else:
        ref = np.concatenate([orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, num_phi, [j], cfg.tol, cfg.max_iter)[0]
                              for j in range(num_phi)])
    assert_rows_match(orc, roots.cpu().numpy(), ref)
    w_ref = orc.caustics(xy, m, cfg.kappa_s, cfg.gamma, ref)
    g, w = roots.cpu().numpy(), caus.cpu().numpy()
    for j in range(num_phi):
        assert_caustics_match(g[j], w[j], ref[j], w_ref[j])
    c2 = api.caustics(dxy, dm, cfg.kappa_s, cfg.gamma, roots)
    assert float((caus - c2).abs().max()) <= 1e-11
    tiled, _, _, st1 = api.critical_curves_ex(dxy, dm, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter,
                                              opt=api.options(regime=1, num_subchains=nsub))
    assert st1.regime == 1
    err, bij = api.match_root_sets(roots, tiled, 1e-10)
    assert bool(bij.all())


@pytest.mark.parametrize("regime,N,num_phi", [(1, 300, 24), (2, 300, 24), (1, 2500, 6)])
def test_equal_mass_fields_take_the_lighter_pair_body(api, orc, regime, N, num_phi):
    """A field whose stars all have the mass m0 runs the equal-mass pair body (unweighted sums scaled by m0 at the end,
    star_sums.cuh).  m0 = 2.5 (not 1, so the scaling is not the identity), both regimes, roots and fused caustic points
    against the oracle; one star made heavier switches back to the general body with the same contract."""
    cfg = CONFIGS["cfg2"]
    xy, _, R = orc.star_field(3, N, cfg.kappa_star, 0, None)
    for m in (np.full(N, 2.5), np.concatenate([np.full(N - 1, 2.5), [2.75]])):
        roots, caus, it, un, st = api.curves_and_caustics(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi, cfg.tol,
                                                          cfg.max_iter, opt=api.options(regime=regime))
        assert st.regime == regime and int(un.sum()) == 0
        ref = np.concatenate([orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, num_phi, [j], cfg.tol, cfg.max_iter)[0]
                              for j in range(num_phi)])
        assert_rows_match(orc, roots.cpu().numpy(), ref)
        w_ref = orc.caustics(xy, m, cfg.kappa_s, cfg.gamma, ref)
        g, w = roots.cpu().numpy(), caus.cpu().numpy()
        for j in range(num_phi):
            assert_caustics_match(g[j], w[j], ref[j], w_ref[j])
        certify_every_row(api, dev(xy), dev(m), cfg, roots)


def test_predictor_order_is_chosen_root_by_root(api, orc):
    """DESIGN.md R18: the extrapolation order is capped by the option and chosen per root from the size of the backward
    differences.  What can be observed through the C-ABI: any cap gives the oracle's root sets; a higher cap never
    costs root-iterations on a smooth grid; and a grid coarse enough that two chains come close (cfg1 at 50 phases,
    2 pi / 50 per row) still converges everywhere with the highest cap, within a few iterations per row."""
    cfg = CONFIGS["cfg2"]
    xy, m, R = field(orc, cfg)
    dxy, dm = dev(xy), dev(m)
    num_phi = 600
    ref, _, _ = orc.critical_curves(xy, m, cfg.kappa_s, cfg.gamma, num_phi)
    work = {}
    for cap in (0, 2, 5, 8):
        r, it, un, st = api.critical_curves_ex(dxy, dm, cfg.kappa_s, cfg.gamma, num_phi,
                                               opt=api.options(predictor_order=cap, num_subchains=2, regime=1))
        assert int(un.sum()) == 0 and st.predictor_order == cap
        assert_rows_match(orc, r.cpu().numpy(), ref)
        work[cap] = st.root_iterations
    assert work[8] <= work[5] <= work[2] <= work[0]
    with pytest.raises(api.MlccError):
        api.critical_curves_ex(dxy, dm, cfg.kappa_s, cfg.gamma, 8, opt=api.options(predictor_order=9))
    c1 = CONFIGS["cfg1"]
    xy1, m1, _ = field(orc, c1)
    for regime in (1, 2):
        r, it, un, st = api.critical_curves_ex(dev(xy1), dev(m1), c1.kappa_s, c1.gamma, 50,
                                               opt=api.options(num_subchains=1, regime=regime))
        ref1, _, _ = orc.critical_curves(xy1, m1, c1.kappa_s, c1.gamma, 50)
        assert int(un.sum()) == 0 and int(it.max()) <= 12
        assert_rows_match(orc, r.cpu().numpy(), ref1)


@pytest.mark.parametrize("max_iter", [1, 2, 3, 6])
def test_tiled_regime_iteration_cap_and_many_subchains(api, orc, max_iter):
    """The tiled regime's driver (rows of several steps in flight at once: DESIGN.md "Driver") at its edges: an iteration
    cap that stops rows early -- every row reports its own count of unfrozen roots, everything is written and finite,
    the call says NOT_CONVERGED -- and plans with so many sub-chains that only two generations, or one (lock-step), of
    slots fit: same root sets as the oracle."""
    cfg = CONFIGS["cfg2"]
    xy, m, R = field(orc, cfg)
    dxy, dm = dev(xy), dev(m)
    num_phi = 96
    r, it, un, st = api.critical_curves_ex(dxy, dm, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, max_iter,
                                           opt=api.options(regime=1, num_subchains=3), strict=False)
    assert st.regime == 1 and bool(torch.isfinite(r).all())
    assert st.status == api.MLCC_ERR_NOT_CONVERGED and st.unconverged_rows == int((un > 0).sum()) > 0
    assert int(it.max()) == max_iter and int(it.min()) >= 1
    again, it2, un2, _ = api.critical_curves_ex(dxy, dm, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, max_iter,
                                                opt=api.options(regime=1, num_subchains=3), strict=False)
    assert torch.equal(again, r) and torch.equal(it2, it) and torch.equal(un2, un)
    if max_iter == 6:
        ref, _, _ = orc.critical_curves(xy, m, cfg.kappa_s, cfg.gamma, 1100)
        for nsub in (200, 400, 512):        # 3, 2 and 1 generations of slots
            full, itf, unf, stf = api.critical_curves_ex(dxy, dm, cfg.kappa_s, cfg.gamma, 1100,
                                                         opt=api.options(regime=1, num_subchains=nsub))
            assert stf.subchains == nsub and int(unf.sum()) == 0
            assert_rows_match(orc, full.cpu().numpy(), ref)
            certify_every_row(api, dxy, dm, cfg, full)


def test_random_shapes_both_regimes_certified_and_against_oracle(api, orc):
    """48 seeded random problems (N 1..300, 1..700 phases, plans from one sub-chain to one per row, every option that
    keeps the root sets): the tiled regime is reproducible bit for bit, every row passes the det J and Vieta
    certificates, the chain regime finds the same root sets, and where the oracle finishes at once (N <= 64,
    <= 64 phases) so does the oracle."""
    rng = np.random.default_rng(20250602)
    with_oracle = stuck = 0
    for case in range(48):
        N = int(rng.choice([1, 2, 3, 5, 17, 40, 64, 100, 129, 200, 257, 300]))
        num_phi = int(rng.choice([1, 2, 3, 7, 16, 33, 64, 100, 257, 400, 700]))
        kappa_star, kappa_s, gamma = rng.uniform(0.05, 0.6), rng.uniform(0.0, 0.6), rng.uniform(-0.6, 0.6)
        nsub = min(int(rng.choice([0, 0, 1, 2, 3, 5, 8, 50, 170, 200, 342, 400, 512])), num_phi)
        kw = [dict(), dict(trust_predictor=1), dict(star_sum_mode=api.MLCC_STAR_SUMS_FMM), dict(aberth_sum_precision=32),
              dict(predictor_order=int(rng.integers(0, 9))),
              dict(trust_predictor=1, star_sum_mode=api.MLCC_STAR_SUMS_FMM)][int(rng.integers(0, 6))]
        what = (case, N, num_phi, nsub, kw)
        xy, m, R = orc.star_field(int(rng.integers(0, 1 << 30)), N, kappa_star, int(rng.integers(0, 2)), None)
        dxy, dm = dev(xy), dev(m)
        opt = api.options(regime=1, num_subchains=nsub, **kw)
        r1, c1, it1, un1, st1 = api.curves_and_caustics(dxy, dm, kappa_s, gamma, num_phi, 1e-12, 60, opt=opt, strict=False)
        r2, c2, it2, un2, _ = api.curves_and_caustics(dxy, dm, kappa_s, gamma, num_phi, 1e-12, 60, opt=opt, strict=False)
        assert torch.equal(r1, r2) and torch.equal(c1, c2) and torch.equal(it1, it2) and torch.equal(un1, un2), what
        if st1.status == api.MLCC_ERR_NOT_CONVERGED:
            # DESIGN.md R6: one star makes F real in z - z_1, the seeds z_1 +- 1 are real, and where the two roots are
            # imaginary (phi = 0 with |gamma| > 1 - kappa_s) the iterates never leave the axis.  The oracle, which
            # follows the paper's seeds too, must fail on the same rows, and so must the chain regime.
            assert N == 1, what
            _, _, un_ref = orc.critical_curves(xy, m, kappa_s, gamma, num_phi, 1e-12, 60)
            assert np.array_equal(un1.cpu().numpy() > 0, un_ref > 0), what
            _, _, _, un3, st3 = api.curves_and_caustics(dxy, dm, kappa_s, gamma, num_phi, 1e-12, 60, strict=False,
                                                        opt=api.options(regime=2, num_subchains=nsub))
            assert st3.status == api.MLCC_ERR_NOT_CONVERGED and torch.equal(un3 > 0, un1 > 0), what
            stuck += 1
            continue
        assert st1.regime == 1 and st1.unconverged_rows == 0 and int(it1.min()) >= 1, what
        assert bool(torch.isfinite(r1).all()) and bool(torch.isfinite(c1).all()), what
        row_newton, row_detj, _ = api.detj_residuals(dxy, dm, kappa_s, gamma, r1)
        assert float(row_detj.max()) <= 1.0 and float(row_newton.max()) <= 1e-10, what
        e1, e2 = api.vieta_residuals(dxy, dm, kappa_s, gamma, r1)
        assert float(e1.max()) <= 1e-11 and float(e2.max()) <= 1e-11, what
        r3, _, _, _, st3 = api.curves_and_caustics(dxy, dm, kappa_s, gamma, num_phi, 1e-12, 60,
                                                   opt=api.options(regime=2, num_subchains=nsub))
        err, bij = api.match_root_sets(r1, r3, ROOT_TOL)
        assert st3.regime == 2 and bool(bij.all()), (what, float(err.max()))
        if N <= 64 and num_phi <= 64:
            ref = orc.critical_curves(xy, m, kappa_s, gamma, num_phi, 1e-12, 80)[0]
            assert_rows_match(orc, r1.cpu().numpy(), ref)
            with_oracle += 1
    assert with_oracle >= 8 and stuck <= 2


def test_chain_regime_limits_and_reports(api, orc):
    """What the chain regime refuses (fields beyond shared memory, far-field sums, a sheet polynomial, the FP32 Aberth
    sum when forced), what AUTO then does, and its max_iter / NaN reports."""
    cfg = CONFIGS["cfg2"]
    xy, m, R = field(orc, cfg)
    dxy, dm = dev(xy), dev(m)
    for bad in (dict(star_sum_mode=api.MLCC_STAR_SUMS_FMM), dict(trust_predictor=1), dict(aberth_sum_precision=32)):
        with pytest.raises(api.MlccError):
            api.critical_curves_ex(dxy, dm, cfg.kappa_s, cfg.gamma, 16, opt=api.options(regime=2, **bad))
        _, _, _, st = api.critical_curves_ex(dxy, dm, cfg.kappa_s, cfg.gamma, 16, opt=api.options(**bad))
        assert st.regime == 1                                       # AUTO falls back to the tiled regime
    big = CONFIGS["cfg3"]
    bxy, bm, _ = field(orc, big)
    with pytest.raises(api.MlccError):
        api.critical_curves_ex(dev(bxy), dev(bm), big.kappa_s, big.gamma, 4, opt=api.options(regime=2))
    # max_iter: unconverged roots are counted per row, everything is written, the status says so
    r, it, un, st = api.critical_curves_ex(dxy, dm, cfg.kappa_s, cfg.gamma, 40, cfg.tol, 2, opt=api.options(regime=2),
                                           strict=False)
    assert st.status == api.MLCC_ERR_NOT_CONVERGED and st.unconverged_rows > 0 and int(un.max()) > 0
    assert int(it.max()) == 2 and bool(torch.isfinite(r).all())
    assert st.unconverged_rows == int((un > 0).sum())
    # an initial guess that sits on a star gives a NaN step: frozen and reported, nothing hangs
    init = torch.cat([dxy, dxy]).contiguous()
    r, it, un, st = api.critical_curves_ex(dxy, dm, cfg.kappa_s, cfg.gamma, 8, cfg.tol, cfg.max_iter,
                                           opt=api.options(regime=2), init_roots=init, strict=False)
    assert st.status == api.MLCC_ERR_DEGENERATE and st.degenerate_roots > 0


# ---------------------------------------------------------------------------------------------
# options do not change the answer (the iteration path is not part of the contract)
# ---------------------------------------------------------------------------------------------
def test_options_do_not_change_the_root_sets(api, orc):
    cfg = CONFIGS["cfg2"]
    xy, m, R = field(orc, cfg)
    num_phi = 240
    ref, _, _ = orc.critical_curves(xy, m, cfg.kappa_s, cfg.gamma, num_phi)
    dxy, dm = dev(xy), dev(m)
    seen_iters = {}
    for regime in (1, 2):
        for order in (0, 1, 2, 3, 5, 8):
            for nsub in (1, 3, 16):
                r, it, un, st = api.critical_curves_ex(dxy, dm, cfg.kappa_s, cfg.gamma, num_phi,
                                                       opt=api.options(num_subchains=nsub, predictor_order=order,
                                                                       regime=regime))
                assert st.subchains == nsub and st.predictor_order == order and int(un.sum()) == 0
                assert st.regime == regime
                assert_rows_match(orc, r.cpu().numpy(), ref)
                seen_iters[(regime, order, nsub)] = st.root_iterations
        # the predictor only removes work
        assert seen_iters[(regime, 3, 1)] < seen_iters[(regime, 0, 1)]
    for T in (1, 2, 4, 8, 16, 32, 64, 128):
        for prec in (32, 64):
            r, it, un, st = api.critical_curves_ex(dxy, dm, cfg.kappa_s, cfg.gamma, num_phi,
                                                   opt=api.options(num_subchains=4, min_lanes_per_root=T,
                                                                   aberth_sum_precision=prec))
            assert st.aberth_sum_precision == prec
            assert_rows_match(orc, r.cpu().numpy(), ref)


@pytest.mark.parametrize("name,num_phi", [("cfg1", 1000), ("cfg2", 400), ("cfg3", 24)])
def test_aberth_sum_precision_changes_the_path_not_the_roots(api, orc, name, num_phi):
    """DESIGN.md reading R19: A = sum 1/(z_k - z_r) multiplies F in the denominator of the update, so its
    arithmetic (double-single FP32 or FP64 seed) may change iteration counts but not the fixed point."""
    cfg = CONFIGS[name]
    xy, m, R = field(orc, cfg)
    rows = np.arange(num_phi)
    ref, _, un = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, num_phi, rows, cfg.tol, cfg.max_iter)
    assert un.sum() == 0
    out = {}
    for prec in (32, 64):
        r, it, unc, st = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi, cfg.tol,
                                                cfg.max_iter, opt=api.options(aberth_sum_precision=prec, regime=1))
        assert int(unc.sum()) == 0 and st.aberth_sum_precision == prec and st.regime == 1
        assert_rows_match(orc, r.cpu().numpy(), ref)
        out[prec] = (r, st)
    # the two paths agree with each other far inside the tolerance, and cost about the same work
    err, bij = api.match_root_sets(out[32][0], out[64][0], 1e-13)
    assert bool(bij.all())
    assert abs(out[32][1].root_iterations - out[64][1].root_iterations) <= 0.02 * out[64][1].root_iterations


@pytest.mark.parametrize("name,num_phi", [("cfg1", 1000), ("cfg2", 4000), ("cfg3", 16)])
def test_fused_curves_and_caustics(api, orc, name, num_phi):
    """mlcc_curves_and_caustics: same roots as mlcc_critical_curves_ex bit for bit; its caustic points
    against the oracle's (1e-9) and against the stand-alone caustic kernel on the same roots."""
    cfg = CONFIGS[name]
    xy, m, R = field(orc, cfg)
    dxy, dm = dev(xy), dev(m)
    roots, caus, iters, unconv, st = api.curves_and_caustics(dxy, dm, cfg.kappa_s, cfg.gamma, num_phi,
                                                             cfg.tol, cfg.max_iter)
    assert int(unconv.sum()) == 0 and st.degenerate_roots == 0
    plain, it2, un2, st2 = api.critical_curves_ex(dxy, dm, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter)
    assert torch.equal(plain, roots) and torch.equal(iters, it2)
    w_kernel = api.caustics(dxy, dm, cfg.kappa_s, cfg.gamma, roots)
    scale = 1 + float(w_kernel.abs().max())
    assert float((caus - w_kernel).abs().max()) <= 1e-12 * scale
    rows = np.arange(num_phi) if cfg.N <= 200 else np.array([0, num_phi // 2, num_phi - 1])
    step = max(1, len(rows) // 100)
    rows = rows[::step]
    ref, _, un = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, num_phi, rows, cfg.tol, cfg.max_iter)
    w_ref = orc.caustics(xy, m, cfg.kappa_s, cfg.gamma, ref)
    g, w = roots.cpu().numpy(), caus.cpu().numpy()
    for i, j in enumerate(rows):
        assert_caustics_match(g[j], w[j], ref[i], w_ref[i])


def test_phase_offset_selects_rows_of_a_larger_grid(api, orc):
    """Rows [off, off+n) of a num_phi_total grid: the multi-GPU sharding contract."""
    cfg = CONFIGS["cfg1"]
    xy, m, R = field(orc, cfg)
    total, off, n = 1000, 300, 120
    ref, _, _ = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, total, np.arange(off, off + n))
    r, it, un, st = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, n,
                                           opt=api.options(phi_index_offset=off, phi_index_total=total))
    assert_rows_match(orc, r.cpu().numpy(), ref)


def test_init_roots_replace_the_cold_seeds(api, orc):
    # one star with gamma > 1 - kappa_s at phi = 0: z_i +/- 1 stay on the real axis for ever
    # (reading R6); rotated seeds converge to +/- i sqrt(m / (gamma - (1 - kappa_s)))
    xy = np.array([[0.0, 0.0]])
    m = np.array([1.0])
    ks, g = 0.5, 0.8
    init = np.array([[np.cos(0.3), np.sin(0.3)], [-np.cos(0.3), -np.sin(0.3)]])
    r, it, un, st = api.critical_curves_ex(dev(xy), dev(m), ks, g, 1, init_roots=dev(init),
                                           opt=api.options(num_subchains=1))
    z = cplx(r.cpu().numpy())[0]
    want = np.sqrt(1.0 / c_phi(ks, g, 0.0) + 0j)
    assert min(abs(z[0] - want), abs(z[0] + want)) < 1e-14 and abs(z[0] + z[1]) < 1e-14
    oref, _, _ = orc.critical_curve_rows(xy, m, ks, g, 1, [0], init_roots=init)
    assert_rows_match(orc, r.cpu().numpy(), oref)


# ---------------------------------------------------------------------------------------------
# degenerate and edge cases
# ---------------------------------------------------------------------------------------------
def test_smallest_problem_single_star_single_phase(api, orc):
    xy = np.array([[0.3, -0.2]])
    m = np.array([1.7])
    r, it, un, st = api.critical_curves_ex(dev(xy), dev(m), 0.1, 0.2, 1)
    ref, _, _ = orc.critical_curves(xy, m, 0.1, 0.2, 1)
    assert r.shape == (1, 2, 2)
    assert_rows_match(orc, r.cpu().numpy(), ref)
    w = api.caustics(dev(xy), dev(m), 0.1, 0.2, r).cpu().numpy()
    assert np.abs(np.sort_complex(cplx(w)[0]) - np.sort_complex(cplx(orc.caustics(xy, m, 0.1, 0.2, ref))[0])).max() < 1e-12


def test_ragged_sizes_span_tiles(api, orc):
    """N chosen so that stars and roots straddle the 256-star shared-memory stages with a ragged tail."""
    for N, num_phi in ((513, 7), (1025, 5), (37, 33), (255, 9), (256, 9), (257, 9)):
        xy, m, R = orc.star_field(11, N, 0.35, 1)
        ref, _, un = orc.critical_curves(xy, m, 0.05, 0.3, num_phi)
        assert un.sum() == 0
        for regime in (1, 2):        # the tiled kernel's stages, and the chain regime that AUTO picks at these sizes
            r, it, unc, st = api.critical_curves_ex(dev(xy), dev(m), 0.05, 0.3, num_phi, opt=api.options(regime=regime))
            assert st.regime == regime
            assert_rows_match(orc, r.cpu().numpy(), ref)
        pts = np.random.default_rng(N).normal(size=(777, 2)) * R
        w = api.caustics(dev(xy), dev(m), 0.05, 0.3, dev(pts)).cpu().numpy()
        wr = orc.caustics(xy, m, 0.05, 0.3, pts)
        assert np.abs(w - wr).max() <= 1e-12 * (1 + np.abs(wr).max())


def test_max_iter_reports_unconverged_but_writes_everything(api, orc):
    cfg = CONFIGS["cfg2"]
    xy, m, R = field(orc, cfg)
    r, it, un, st = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, 8, max_iter=2,
                                           opt=api.options(num_subchains=1), strict=False)
    assert st.status == api.MLCC_ERR_NOT_CONVERGED and st.unconverged_rows >= 1
    assert int(un.max()) > 0 and int(it.max()) == 2
    assert torch.isfinite(r).all()
    with pytest.raises(api.MlccError) as e:
        api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, 8, max_iter=2)
    assert e.value.status == api.MLCC_ERR_NOT_CONVERGED
    # the oracle agrees on which rows are unfinished after 2 sweeps of the cold row
    _, it_o, un_o = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, 8, [4], max_iter=2)
    assert un_o[0] > 0 and it_o[0] == 2 and int(un[4]) == int(un_o[0])


def test_coincident_stars_are_reported_degenerate(api):
    xy = np.array([[0.5, 0.5], [0.5, 0.5], [-1.0, 0.2]])
    m = np.ones(3)
    # two stars at one point: P(z) has only 2N - 2 roots, the degree claim fails
    with pytest.raises(api.MlccError) as e:
        api.critical_curves_ex(dev(xy), dev(m), 0.0, 0.1, 4)
    assert e.value.status == api.MLCC_ERR_DEGENERATE
    xy[1, 0] = np.nan
    with pytest.raises(api.MlccError) as e:
        api.critical_curves_ex(dev(xy), dev(m), 0.0, 0.1, 4)
    assert e.value.status == api.MLCC_ERR_INVALID_ARG


def test_empty_inputs(api):
    xy, m = dev(np.zeros((2, 2))), dev(np.ones(2))
    empty = torch.empty((0, 2), dtype=torch.float64, device="cuda")
    assert api.caustics(xy, m, 0.0, 0.1, empty).shape == (0, 2)
    e, b = api.match_root_sets(torch.empty((0, 5, 2), dtype=torch.float64, device="cuda"),
                               torch.empty((0, 5, 2), dtype=torch.float64, device="cuda"), 1e-10)
    assert e.shape == (0,) and b.shape == (0,)


def test_binding_rejects_cpu_tensors(api):
    with pytest.raises(TypeError):
        api.caustics(torch.zeros(2, 2, dtype=torch.float64), torch.ones(2, dtype=torch.float64).cuda(), 0, 0.1,
                     torch.zeros(3, 2, dtype=torch.float64).cuda())


# ---------------------------------------------------------------------------------------------
# a8 validator against the oracle's brute force
# ---------------------------------------------------------------------------------------------
def test_match_root_sets_against_brute_force(api, orc):
    rng = np.random.default_rng(3)
    for S, n in ((5, 1), (7, 2), (6, 40), (3, 1000), (3, 20011)):
        b = rng.normal(size=(S, n, 2)) * 50
        a = np.empty_like(b)
        for s in range(S):
            a[s] = b[s][rng.permutation(n)] + rng.normal(size=(n, 2)) * 1e-12
        if n >= 40:
            a[0, 3] = a[0, 5]            # duplicated root, one missing
            a[1, 0, 0] += 1e-3           # beyond tolerance
            a[2, 7] += 30.0              # far from everything: exercises the ring expansion / fallback
        e_o, b_o = orc.match_root_sets(a, b, 1e-10)
        e_g, b_g = api.match_root_sets(dev(a), dev(b), 1e-10)
        assert b_g.cpu().numpy().tolist() == b_o.tolist()
        assert np.abs(e_g.cpu().numpy() - e_o).max() <= 1e-15 * (1 + e_o.max())
    # clustered sets with an outlier pair (the shape of a critical-curve row) and a non-finite value
    cfg = CONFIGS["cfg2"]
    xy, m, R = field(orc, cfg)
    ref, _, _ = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, 16, np.arange(4))
    a = ref[:, rng.permutation(ref.shape[1])] + 1e-13
    e_o, b_o = orc.match_root_sets(a, ref, 1e-10)
    e_g, b_g = api.match_root_sets(dev(a), dev(ref), 1e-10)
    assert b_o.all() and b_g.cpu().numpy().all() and np.abs(e_g.cpu().numpy() - e_o).max() < 1e-18
    a[1, 2, 0] = np.nan
    e_g, b_g = api.match_root_sets(dev(a), dev(ref), 1e-10)
    assert b_g.cpu().numpy().tolist() == [1, 0, 1, 1] and np.isinf(e_g.cpu().numpy()[1])


# ---------------------------------------------------------------------------------------------
# host-buffer entry points
# ---------------------------------------------------------------------------------------------
def test_host_buffer_entry_points(api, orc):
    cfg = CONFIGS["cfg1"]
    xy, m, R = field(orc, cfg)
    roots_h, caus_h, st = api.curves_and_caustics_host(xy, m, cfg.kappa_s, cfg.gamma, 200)
    ref, _, _ = orc.critical_curves(xy, m, cfg.kappa_s, cfg.gamma, 200)
    assert_rows_match(orc, roots_h, ref)
    ref_caus = orc.caustics(xy, m, cfg.kappa_s, cfg.gamma, ref)
    for j in range(0, 200, 7):
        assert_caustics_match(roots_h[j], caus_h[j], ref[j], ref_caus[j])
    r2 = api.critical_curves_host(xy, m, cfg.kappa_s, cfg.gamma, 200)
    assert np.array_equal(r2, roots_h)
    c2 = api.caustics_host(xy, m, cfg.kappa_s, cfg.gamma, ref)
    assert np.abs(c2 - orc.caustics(xy, m, cfg.kappa_s, cfg.gamma, ref)).max() < 1e-12


@pytest.mark.parametrize("name,num_phi,subchains", [("cfg1", 1000, 0), ("cfg2", 4000, 0), ("cfg2", 1501, 5),
                                                    ("cfg3", 640, 0), ("cfg3", 97, 1)])
def test_host_entry_point_with_pinned_outputs_copies_rows_while_solving(api, orc, name, num_phi, subchains):
    """Pinned host outputs get the finished rows on a second stream while the solve runs (pageable ones are copied
    once at the end).  Both must deliver, in every row, exactly the bits the device path computes; sentinel values in
    the destination show that no row is left out, whatever the sub-chain layout and the number of polls."""
    cfg = CONFIGS[name]
    xy, m, R = field(orc, cfg)
    opt = api.options(num_subchains=subchains)
    d_roots, d_caus, _, _, st = api.curves_and_caustics(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi, cfg.tol,
                                                        cfg.max_iter, opt=opt)
    n_r = 2 * cfg.N
    p_roots = torch.full((num_phi, n_r, 2), float("nan"), dtype=torch.float64).pin_memory()
    p_caus = torch.full((num_phi, n_r, 2), float("nan"), dtype=torch.float64).pin_memory()
    api.curves_and_caustics_host(xy, m, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter, opt=opt,
                                 out_roots=p_roots, out_caustics=p_caus)
    assert torch.equal(p_roots, d_roots.cpu()) and torch.equal(p_caus, d_caus.cpu())
    n_roots, n_caus, _ = api.curves_and_caustics_host(xy, m, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter,
                                                      opt=opt)                      # pageable numpy outputs
    assert np.array_equal(n_roots, p_roots.numpy()) and np.array_equal(n_caus, p_caus.numpy())
    # roots only, pinned
    p_only = torch.full((num_phi, n_r, 2), float("nan"), dtype=torch.float64).pin_memory()
    api.curves_and_caustics_host(xy, m, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter, opt=opt,
                                 out_roots=p_only, want_caustics=False)
    assert torch.equal(p_only, p_roots)
    ref_rows = [0, num_phi // 2, num_phi - 1]
    ref, _, un = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, num_phi, ref_rows[:1], cfg.tol, cfg.max_iter)
    assert_rows_match(orc, p_roots.numpy()[:1], ref)


def test_fp64_peak_probe_is_plausible(api):
    tf = api.fp64_peak(20.0)
    assert 5.0 < tf < 80.0, tf


# ---------------------------------------------------------------------------------------------
# far-field split of the star sums (Section 4.1)
# ---------------------------------------------------------------------------------------------
def _points_for_star_sums(xy, R, n, seed):
    """Points shaped like critical points: most within ~1 Einstein radius of a star, some anywhere in the field,
    a few outside the stars' bounding square (the outer root pair) and on the grid's edge."""
    rng = np.random.default_rng(seed)
    near = xy[rng.integers(0, len(xy), n)] + rng.normal(size=(n, 2)) * 0.7
    anywhere = rng.uniform(-R, R, size=(n // 2, 2))
    outside = rng.normal(size=(16, 2))
    outside = outside / np.linalg.norm(outside, axis=1, keepdims=True) * R * rng.uniform(1.5, 3.0, size=(16, 1))
    corner = np.array([[xy[:, 0].min(), xy[:, 1].min()], [xy[:, 0].max(), xy[:, 1].max()],
                       [xy[:, 0].max() + 1e-9, 0.0], [0.0, xy[:, 1].min() - 1e-9]])
    return np.concatenate([near, anywhere, outside, corner])


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg4"])
def test_star_sums_direct_and_fmm_against_oracle(api, orc, name):
    """mlcc_star_sums in both modes against the oracle's long-double straight sums.  Tolerance: the sums are
    N terms of size ~ m/d^k accumulated in FP64, so 1e-12 relative to sum |term| is ~100 ulp-sums; the split's
    truncation (rho^32 = 3e-18) must not show at that level."""
    cfg = CONFIGS[name]
    xy, m, R = field(orc, cfg)
    pts = _points_for_star_sums(xy, R, 600, cfg.N)
    ref = orc.star_sums(xy, m, pts, long_double=True)
    z = pts[:, 0] + 1j * pts[:, 1]
    d = np.abs(z[:, None] - (xy[:, 0] + 1j * xy[:, 1])[None, :])
    scale = np.stack([(1 / d).sum(1), (m / d ** 2).sum(1), (m / d ** 3).sum(1), (m / d).sum(1)], axis=1)
    scale = np.repeat(scale, 2, axis=1)
    for mode in (api.MLCC_STAR_SUMS_DIRECT, api.MLCC_STAR_SUMS_FMM):
        got = api.star_sums(dev(xy), dev(m), dev(pts), mode=mode).cpu().numpy()
        assert np.isfinite(got).all()
        assert (np.abs(got - ref) / scale).max() < 1e-12, (mode, (np.abs(got - ref) / scale).max())


def test_fmm_truncation_follows_the_geometric_bound(api, orc):
    """Order p leaves an error below C rho^(p+1), rho = (1/sqrt 2)/2.5 = 0.283: each
    8 more terms must gain ~4 decimal digits until FP64 rounding is reached.  Also other node sizes."""
    cfg = CONFIGS["cfg3"]
    xy, m, R = field(orc, cfg)
    pts = _points_for_star_sums(xy, R, 400, 5)[:600]          # inside points only matter here
    ref = orc.star_sums(xy, m, pts, long_double=True)
    errs = {}
    for order in (7, 15, 23, 31):
        got = api.star_sums(dev(xy), dev(m), dev(pts), mode=api.MLCC_STAR_SUMS_FMM, fmm_order=order).cpu().numpy()
        errs[order] = np.abs(got[:, 2:4] - ref[:, 2:4]).max()   # S2: the sum that carries F
    rho = (0.5 ** 0.5) / 2.5
    total = float((m[None, :] / 1.0).sum())                     # crude constant: sum m_i / s^2 with s >= 1
    for order, e in errs.items():
        assert e < max(total * (order + 1) * rho ** (order + 1), 1e-11), (order, e)
    assert errs[15] < 1e-3 * errs[7] and (errs[23] < 1e-2 * errs[15] or errs[23] < 1e-11)
    assert errs[31] < 1e-11
    for spn in (1, 2, 16, 64, 100000):
        got = api.star_sums(dev(xy), dev(m), dev(pts), mode=api.MLCC_STAR_SUMS_FMM, fmm_stars_per_node=spn).cpu().numpy()
        assert np.abs(got - ref).max() < 1e-9 * (1 + np.abs(ref).max())


@pytest.mark.parametrize("name,num_phi", [("cfg1", 1000), ("cfg2", 4000), ("cfg3", 64)])
def test_fmm_mode_gives_the_same_root_sets_and_caustics(api, orc, name, num_phi):
    cfg = CONFIGS[name]
    xy, m, R = field(orc, cfg)
    rows = np.arange(num_phi) if cfg.N <= 200 else np.array([0, 1, num_phi // 2, num_phi - 1])
    ref, _, un = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, num_phi, rows, cfg.tol, cfg.max_iter)
    assert un.sum() == 0
    w_ref = orc.caustics(xy, m, cfg.kappa_s, cfg.gamma, ref)
    for prec in (32, 64):
        opt = api.options(star_sum_mode=api.MLCC_STAR_SUMS_FMM, aberth_sum_precision=prec)
        roots, caus, iters, unconv, st = api.curves_and_caustics(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi,
                                                                 cfg.tol, cfg.max_iter, opt=opt)
        assert int(unconv.sum()) == 0 and st.degenerate_roots == 0
        g, w = roots.cpu().numpy(), caus.cpu().numpy()
        assert_rows_match(orc, g[rows], ref)
        for i, j in enumerate(rows[::max(1, len(rows) // 50)]):
            ii = i * max(1, len(rows) // 50)
            assert_caustics_match(g[j], w[j], ref[ii], w_ref[ii])
        # against the direct mode of the same library: far inside the parity tolerance
        plain, _, _, _ = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi, cfg.tol,
                                                cfg.max_iter, opt=api.options(aberth_sum_precision=prec))
        err, bij = api.match_root_sets(roots, plain, 1e-12)
        assert bool(bij.all())
        # reproducible
        r2, _, _, _, _ = api.curves_and_caustics(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi, cfg.tol,
                                                 cfg.max_iter, opt=opt)
        assert torch.equal(r2, roots)


def test_fmm_mode_full_size_cfg4_sampled_rows(api, orc):
    cfg = CONFIGS["cfg4"]
    xy, m, R = field(orc, cfg)
    num_phi = 512
    opt = api.options(star_sum_mode=api.MLCC_STAR_SUMS_FMM)
    roots, iters, unconv, st = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi, cfg.tol,
                                                      cfg.max_iter, opt=opt)
    assert int(unconv.sum()) == 0 and st.degenerate_roots == 0
    e1, e2 = vieta_all_rows(roots, xy, m, cfg.kappa_s, cfg.gamma, num_phi)
    assert e1 < 1e-12 and e2 < 1e-12, (e1, e2)
    for j in (0, 255):
        ref, _, un = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, num_phi, [j], cfg.tol, cfg.max_iter)
        assert un.sum() == 0
        assert_rows_match(orc, roots[j:j + 1].cpu().numpy(), ref)
    check_row_invariants(orc, xy, m, cfg.kappa_s, cfg.gamma, 100, num_phi, cplx(roots[100].cpu().numpy()))


# ---------------------------------------------------------------------------------------------
# chain joining and the caustic-crossing map
# ---------------------------------------------------------------------------------------------
def _map_window(caus, n_pix, margin=0.05):
    lo, hi = caus.reshape(-1, 2).min(0), caus.reshape(-1, 2).max(0)
    side = float((hi - lo).max()) * (1 + 2 * margin)
    c = 0.5 * (lo + hi)
    return float(c[0] - side / 2), float(c[1] - side / 2), side / n_pix


@pytest.mark.parametrize("name,num_phi,n_pix", [("cfg1", 1000, 257), ("cfg2", 600, 96)])
def test_link_rows_and_crossing_map_against_oracle(api, orc, name, num_phi, n_pix):
    """GPU roots and caustics -> GPU joining -> GPU map, against the oracle's joining and its per-pixel winding
    numbers of the same points.  Integer outputs: exact, except pixels whose centre the oracle flags as lying on a
    segment to rounding (either neighbour's count is right there)."""
    cfg = CONFIGS[name]
    xy, m, R = field(orc, cfg)
    roots, caus, iters, unconv, st = api.curves_and_caustics(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi,
                                                             cfg.tol, cfg.max_iter)
    assert st.subchains > 1                       # the column order really changes between rows
    nxt, bij = api.link_rows(roots)
    g_roots, g_caus = roots.cpu().numpy(), caus.cpu().numpy()
    o_nxt, o_bij = orc.link_rows(g_roots)
    assert o_bij.all() and bool(bij.all())
    assert np.array_equal(nxt.cpu().numpy(), o_nxt)
    assert (o_nxt != np.arange(o_nxt.shape[1])[None, :]).any()
    x0, y0, pixel = _map_window(g_caus, n_pix)
    got = api.crossing_map(caus, nxt, x0, y0, pixel, n_pix, n_pix).cpu().numpy()
    ref, amb = orc.crossing_map(g_caus, o_nxt, x0, y0, pixel, n_pix, n_pix, want_ambiguous=True)
    assert amb.mean() < 0.01
    assert np.array_equal(got[amb == 0], ref[amb == 0])
    assert ref.min() >= 0 and ref.max() >= 2 and ref[0, 0] == 0      # crossings are counted, never negative
    # a window that cuts the caustics, non-square, off-centre
    got2 = api.crossing_map(caus, nxt, x0 + 0.31 * n_pix * pixel, y0 + 0.4 * n_pix * pixel, pixel * 0.37, 75, 41).cpu().numpy()
    ref2, amb2 = orc.crossing_map(g_caus, o_nxt, x0 + 0.31 * n_pix * pixel, y0 + 0.4 * n_pix * pixel, pixel * 0.37,
                                  75, 41, want_ambiguous=True)
    assert np.array_equal(got2[amb2 == 0], ref2[amb2 == 0])
    # reproducible to the bit
    assert np.array_equal(api.crossing_map(caus, nxt, x0, y0, pixel, n_pix, n_pix).cpu().numpy(), got)


def test_crossing_map_on_oracle_points_and_open_chains(api, orc):
    """Same points on both sides (oracle roots/caustics uploaded): identity columns, then an open set of rows."""
    cfg = CONFIGS["cfg1"]
    xy, m, R = field(orc, cfg)
    num_phi = 360
    roots, _, _ = orc.critical_curves(xy, m, cfg.kappa_s, cfg.gamma, num_phi)
    caus = orc.caustics(xy, m, cfg.kappa_s, cfg.gamma, roots)
    o_nxt, o_bij = orc.link_rows(roots)
    assert o_bij.all()
    nxt, bij = api.link_rows(dev(roots))
    assert np.array_equal(nxt.cpu().numpy(), o_nxt) and bool(bij.all())
    x0, y0, pixel = _map_window(caus, 128)
    ref, amb = orc.crossing_map(caus, o_nxt, x0, y0, pixel, 128, 128, want_ambiguous=True)
    got = api.crossing_map(dev(caus), nxt, x0, y0, pixel, 128, 128).cpu().numpy()
    assert np.array_equal(got[amb == 0], ref[amb == 0])
    # the oracle's rows are one chain per column except at the wrap: next = None is wrong only there
    got_id = api.crossing_map(dev(caus), None, x0, y0, pixel, 128, 128).cpu().numpy()
    ref_id = orc.crossing_map(caus, None, x0, y0, pixel, 128, 128)
    assert (got_id != ref_id).mean() < 0.01
    # open chains (closed = 0): with row 0 appended as an extra last row the open polygons are the closed ones
    ext = np.concatenate([caus, caus[:1]])
    ext_nxt = np.concatenate([o_nxt, np.arange(o_nxt.shape[1], dtype=np.int32)[None, :]])
    open_map = api.crossing_map(dev(ext), dev(ext_nxt, torch.int32), x0, y0, pixel, 128, 128, closed=False).cpu().numpy()
    assert np.array_equal(open_map, got)

def test_link_rows_edge_cases(api, orc):
    rng = np.random.default_rng(8)
    for S, n in ((1, 1), (1, 7), (2, 1), (5, 300), (3, 2500)):
        rows = rng.normal(size=(S, n, 2)) * 20
        nxt, bij = api.link_rows(dev(rows))
        o_nxt, o_bij = orc.link_rows(rows)
        assert np.array_equal(nxt.cpu().numpy(), o_nxt) and bij.cpu().numpy().tolist() == o_bij.tolist()
    rows[1, 3, 0] = np.nan
    nxt, bij = api.link_rows(dev(rows))
    b = bij.cpu().numpy()
    assert b[1] == 0 and b[0] == 0 and (nxt.cpu().numpy()[1] == -1).all()     # rows 0 -> 1 and 1 -> 2 involve the NaN row
    empty = torch.empty((0, 4, 2), dtype=torch.float64, device="cuda")
    n0, b0 = api.link_rows(empty)
    assert n0.shape == (0, 4) and b0.shape == (0,)


# ---------------------------------------------------------------------------------------------
# rectangular microlens field (Appendix A-B)
# ---------------------------------------------------------------------------------------------
def _rect_field(N, kappa_star, aspect, seed):
    """N equal-or-random-mass stars uniform in the rectangle of area pi N / kappa_star (Eq. 9 with sum m = N)."""
    rng = np.random.default_rng(seed)
    c2 = np.sqrt(np.pi * N / (4 * kappa_star * aspect))
    c1 = aspect * c2
    xy = rng.uniform(-1, 1, size=(N, 2)) * [c1, c2]
    m = rng.uniform(0.3, 1.7, size=N)
    m *= N / m.sum()
    return xy, m, c1, c2


@pytest.mark.parametrize("N,aspect,num_phi,t_req", [(12, 1.5, 96, 7), (150, 0.6, 48, 0), (600, 2.0, 10, 0)])
def test_rectangular_field_roots_and_caustics_against_oracle(api, orc, N, aspect, num_phi, t_req):
    """The CUDA path evaluates the sheet as the real-coefficient polynomial of mlcc_rect_sheet; the oracle evaluates
    Eq. B2 / B7 / B9 as printed.  Same 2N + t - 1 roots per row (1e-10 (1 + |z|)), caustic points within 1e-9."""
    kstar, ks, g = 0.4, 0.05, 0.2
    xy, m, c1, c2 = _rect_field(N, kstar, aspect, 17 + N)
    coef, shift, t = api.rect_sheet(kstar, c1, c2, s=1.5, eps=1e-9, t=t_req)
    seed_r = 1.2 * np.hypot(c1, c2)
    n_r = 2 * N + t - 1
    rows = np.arange(num_phi) if N <= 150 else np.array([0, num_phi // 2, num_phi - 1])
    ref, _, un = orc.rect_critical_curve_rows(xy, m, ks, g, kstar, c1, c2, t, seed_r, num_phi, rows)
    assert un.sum() == 0 and ref.shape[1] == n_r
    w_ref = orc.rect_caustics(xy, m, ks, g, kstar, c1, c2, t, ref)
    for mode in (api.MLCC_STAR_SUMS_DIRECT, api.MLCC_STAR_SUMS_FMM):
        opt = api.options(sheet_poly=coef, seed_radius=seed_r, star_sum_mode=mode)
        roots, caus, iters, unconv, st = api.curves_and_caustics(dev(xy), dev(m), ks, g + shift, num_phi, opt=opt)
        assert roots.shape == (num_phi, n_r, 2) and int(unconv.sum()) == 0 and st.degenerate_roots == 0
        gr, gw = roots.cpu().numpy(), caus.cpu().numpy()
        assert_rows_match(orc, gr[rows], ref)
        for i, j in enumerate(rows):
            assert_caustics_match(gr[j], gw[j], ref[i], w_ref[i])
    # the extra roots exist and lie outside the rectangle (where the truncated series stops representing the sheet)
    zr = cplx(ref[0])
    outside = (np.abs(zr.real) > c1) | (np.abs(zr.imag) > c2)
    assert outside.sum() >= t - 1
    # without the polynomial the same stars have 2N roots: the option changes the problem, and is needed
    plain, _, _, _ = api.critical_curves_ex(dev(xy), dev(m), ks, g + shift, num_phi)
    assert plain.shape[1] == 2 * N


def test_rectangular_field_from_the_seeded_generator(api, orc):
    """The whole rectangular path on generated inputs: mlcc_star_field_rect -> mlcc_rect_sheet -> curves and caustics,
    against the oracle on the oracle's own generated field (bit-identical positions)."""
    N, kstar, aspect, ks, g, num_phi = 300, 0.4, 1.6, 0.05, 0.15, 12
    xy, m, c1, c2 = api.star_field_rect(11, N, kstar, aspect, 1)
    oxy, om, oc1, oc2 = orc.star_field_rect(11, N, kstar, aspect, 1)
    assert (c1, c2) == (oc1, oc2) and np.array_equal(xy.cpu().numpy(), oxy)
    coef, shift, t = api.rect_sheet(kstar, c1, c2, s=1.5, eps=1e-9)
    seed_r = 1.2 * np.hypot(c1, c2)
    rows = np.array([0, 5, 11])
    ref, _, un = orc.rect_critical_curve_rows(oxy, om, ks, g, kstar, c1, c2, t, seed_r, num_phi, rows)
    assert un.sum() == 0
    w_ref = orc.rect_caustics(oxy, om, ks, g, kstar, c1, c2, t, ref)
    opt = api.options(sheet_poly=coef, seed_radius=seed_r)
    roots, caus, iters, unconv, st = api.curves_and_caustics(xy, m, ks, g + shift, num_phi, opt=opt)
    assert int(unconv.sum()) == 0 and roots.shape[1] == 2 * N + t - 1
    gr, gw = roots.cpu().numpy(), caus.cpu().numpy()
    assert_rows_match(orc, gr[rows], ref)
    for i, j in enumerate(rows):
        assert_caustics_match(gr[j], gw[j], ref[i], w_ref[i])


def test_rectangular_field_argument_checks(api):
    xy, m = dev(np.array([[0.1, 0.2], [-0.4, 0.3]])), dev(np.ones(2))
    with pytest.raises(api.MlccError) as e:          # extra roots need a seed circle (or init_roots)
        api.critical_curves_ex(xy, m, 0.0, 0.1, 4, opt=api.options(sheet_poly=[0, 0, 0, 0.01], seed_radius=0.0))
    assert e.value.status == api.MLCC_ERR_INVALID_ARG
    with pytest.raises(api.MlccError) as e:          # vanishing leading coefficient: the degree would drop
        api.critical_curves_ex(xy, m, 0.0, 0.1, 4, opt=api.options(sheet_poly=[0, 0, 0, 0.0], seed_radius=2.0))
    assert e.value.status == api.MLCC_ERR_INVALID_ARG
    # degree 1 (H = h1 u) is a pure shear shift: no extra roots, same as gamma - h1
    a, _, _, _ = api.critical_curves_ex(xy, m, 0.0, 0.1, 4, opt=api.options(sheet_poly=[0.0, 0.03]))
    b, _, _, _ = api.critical_curves_ex(xy, m, 0.0, 0.07, 4)
    err, bij = api.match_root_sets(a, b, 1e-12)
    assert a.shape == b.shape and bool(bij.all())


def test_confirm_iterations_without_the_aberth_sum(api, orc):
    """DESIGN.md reading R27: once every step of an iteration was below skip_aberth_sum_below, the next iteration of
    the row leaves A out.  Same root sets (the fixed point F = 0 does not involve A), same iteration counts, fewer
    (root, root) pairs; a negative threshold restores the Aberth sum in every iteration."""
    cfg = CONFIGS["cfg3"]
    xy, m, R = field(orc, cfg)
    num_phi = 400
    rows = np.array([0, 57, 200, 399])
    ref, _, un = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, num_phi, rows, cfg.tol, cfg.max_iter)
    assert un.sum() == 0
    out = {}
    for name, thr in (("default", 0.0), ("never", -1.0), ("loose", 1e-5)):
        for mode in (api.MLCC_STAR_SUMS_DIRECT, api.MLCC_STAR_SUMS_FMM):
            r, it, unc, st = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi, cfg.tol,
                                                    cfg.max_iter, opt=api.options(skip_aberth_sum_below=thr,
                                                                                  star_sum_mode=mode))
            assert int(unc.sum()) == 0 and st.degenerate_roots == 0
            assert_rows_match(orc, r.cpu().numpy()[rows], ref)
            out[(name, mode)] = (r, it, st)
    n_r = 2 * cfg.N
    for mode in (api.MLCC_STAR_SUMS_DIRECT, api.MLCC_STAR_SUMS_FMM):
        never, default, loose = (out[(k, mode)][2] for k in ("never", "default", "loose"))
        assert never.root_pairs == never.root_iterations * (n_r - 1)
        assert default.root_pairs < 0.95 * default.root_iterations * (n_r - 1)
        assert loose.root_pairs <= default.root_pairs
        assert abs(default.root_iterations - never.root_iterations) <= 0.01 * never.root_iterations
        err, bij = api.match_root_sets(out[("default", mode)][0], out[("never", mode)][0], 1e-13)
        assert bool(bij.all())


@pytest.mark.parametrize("name,num_phi", [("cfg1", 1000), ("cfg2", 4000), ("cfg3", 5000)])
def test_trust_predictor_starts_rows_with_newton_steps(api, orc, name, num_phi):
    """DESIGN.md reading R30 (mlcc_options.trust_predictor): rows seeded by the full-order predictor start without the
    Aberth sum; a Newton step above the skip threshold is discarded and the root falls back to Eq. 17.  Same root
    sets as the oracle and as the default path, every row complete (Vieta sums), far fewer (root, root) pairs."""
    cfg = CONFIGS[name]
    xy, m, R = field(orc, cfg)
    rows = np.arange(num_phi) if cfg.N <= 200 else np.array([0, 1, 2, 3, 1249, 2500, 2501, 4999])
    if cfg.N <= 200:
        ref, _, un = orc.critical_curves(xy, m, cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter)
    else:
        ref = np.concatenate([orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, num_phi, [j], cfg.tol,
                                                      cfg.max_iter)[0] for j in rows])
    for mode in (api.MLCC_STAR_SUMS_DIRECT, api.MLCC_STAR_SUMS_FMM):
        base, it0, un0, st0 = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi, cfg.tol,
                                                     cfg.max_iter, opt=api.options(star_sum_mode=mode, regime=1))
        got, it1, un1, st1 = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi, cfg.tol,
                                                    cfg.max_iter, opt=api.options(star_sum_mode=mode, trust_predictor=1))
        assert int(un1.sum()) == 0 and st1.degenerate_roots == 0 and st1.unconverged_rows == 0
        assert_rows_match(orc, got.cpu().numpy()[rows], ref)
        e1, e2 = vieta_all_rows(got, xy, m, cfg.kappa_s, cfg.gamma, num_phi)
        assert e1 < 1e-12 and e2 < 1e-12, (e1, e2)
        err, bij = api.match_root_sets(got, base, 1e-12)
        assert bool(bij.all())
        if name != "cfg1":     # cfg1's grid is coarse (2 pi / 1000): many predictions miss the threshold and fall back
            # what is left are the cold rows (~20 full iterations each), the first rows of every sub-chain and fallbacks
            assert st1.root_pairs < 0.75 * st0.root_pairs, (st1.root_pairs, st0.root_pairs)
            assert st1.root_iterations < 1.35 * st0.root_iterations
        else:
            assert st1.root_iterations < 2.5 * st0.root_iterations
    # fused caustics of the trusted path against the stand-alone kernel on the same roots
    r, c, _, _, st = api.curves_and_caustics(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi, cfg.tol, cfg.max_iter,
                                             opt=api.options(trust_predictor=1))
    c2 = api.caustics(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, r)
    assert float((c - c2).abs().max()) <= 1e-11
    # with the plain previous row as the seed (order 0) nothing is trusted: identical to the default path
    a, _, _, sa = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, min(num_phi, 200), cfg.tol, cfg.max_iter,
                                         opt=api.options(predictor_order=0, trust_predictor=1))
    b, _, _, sb = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, min(num_phi, 200), cfg.tol, cfg.max_iter,
                                         opt=api.options(predictor_order=0, skip_aberth_sum_below=1e-8, regime=1))
    assert torch.equal(a, b) and sa.root_pairs == sb.root_pairs
    with pytest.raises(api.MlccError):
        api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, 8, opt=api.options(trust_predictor=2))


@pytest.mark.parametrize("tol,skip", [(1e-6, 0.0), (1e-6, 1e-9), (1e-12, 1e-13)])
def test_trust_predictor_with_a_skip_threshold_below_tol(api, orc, tol, skip):
    """The guarded first iteration of a trusted row when skip_aberth_sum_below < tol (library default 1e-8 against
    tol = 1e-6, or an explicit threshold below tol): rejected Newton steps between the two thresholds must stay in the
    list -- k_apply's two passes use one predicate (step_kind) -- so no root is left at its predictor seed: every row
    complete (Vieta), every root certified by its Newton residual, none unconverged, sets equal to the oracle's."""
    cfg = CONFIGS["cfg2"]
    xy, m, R = field(orc, cfg)
    num_phi = 1200
    got, it, un, st = api.critical_curves_ex(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, num_phi, tol, cfg.max_iter,
                                             opt=api.options(trust_predictor=1, skip_aberth_sum_below=skip))
    assert int(un.sum()) == 0 and st.unconverged_rows == 0 and st.degenerate_roots == 0
    ref, _, uno = orc.critical_curves(xy, m, cfg.kappa_s, cfg.gamma, num_phi, tol, cfg.max_iter)
    assert uno.sum() == 0
    # a step below tol = 1e-6 was still APPLIED: the error left is of second order in it
    assert_rows_match(orc, got.cpu().numpy(), ref, tol=1e-10 if tol < 1e-9 else 1e-9)
    e1, e2 = vieta_all_rows(got, xy, m, cfg.kappa_s, cfg.gamma, num_phi)
    assert e1 < 1e-9 and e2 < 1e-9, (e1, e2)
    rn, rd, _ = api.detj_residuals(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, got)
    assert float(rn.max()) < (1e-11 if tol < 1e-9 else 1e-9), float(rn.max())


def test_crossing_map_full_size_cfg4_sampled_pixels(api, orc):
    """cfg4 at its full size (10^4 phases x 2*10^4 roots = 2*10^8 caustic segments, far-field star sums for speed):
    chains joined on the GPU, 2048^2 map, and a 4 x 4 sample of its pixels recomputed one by one by the oracle's
    per-pixel winding sum over all segments of the GPU's own caustic points."""
    cfg = CONFIGS["cfg4"]
    xy, m, R = field(orc, cfg)
    opt = api.options(star_sum_mode=api.MLCC_STAR_SUMS_FMM)
    roots, caus, iters, unconv, st = api.curves_and_caustics(dev(xy), dev(m), cfg.kappa_s, cfg.gamma, cfg.num_phi,
                                                             cfg.tol, cfg.max_iter, opt=opt, want_diagnostics=False)
    assert st.unconverged_rows == 0 and st.degenerate_roots == 0
    nxt, bij = api.link_rows(roots)
    n_bad = int((bij == 0).sum())
    assert n_bad <= 5, n_bad                       # rows where two roots are closer than their step in phi (reported)
    n_pix, half = 2048, 30.0
    pixel = 2 * half / n_pix
    cmap = api.crossing_map(caus, nxt, -half, -half, pixel, n_pix, n_pix)
    assert int(cmap.min()) >= -1 and int(cmap.max()) >= 3
    # sample: three pixels of every count 0..3, each recomputed by the oracle as a 1 x 1 map centred on that pixel
    g_caus, g_nxt, g_map = caus.cpu().numpy(), nxt.cpu().numpy(), cmap.cpu().numpy()
    rng = np.random.default_rng(6)
    checked = 0
    for value in range(4):
        iy, ix = np.nonzero(g_map == value)
        assert len(iy) > 0, value
        for q in rng.choice(len(iy), size=3, replace=False):
            x0s, y0s = -half + ix[q] * pixel, -half + iy[q] * pixel
            ref, amb = orc.crossing_map(g_caus, g_nxt, x0s, y0s, pixel, 1, 1, want_ambiguous=True)
            if amb[0, 0]:
                continue
            assert ref[0, 0] == value, (ix[q], iy[q], value, ref[0, 0])
            checked += 1
    assert checked >= 10
