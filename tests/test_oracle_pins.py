"""Pins for the CPU oracle: every check here is against something other than the oracle itself —
closed forms, numpy's companion-matrix eigenvalues of the expanded polynomial, algebraic
invariants of the root set (Vieta), long-double residuals, scipy's assignment solver, analytic
CDFs, published known-answer vectors.  None of this needs a GPU.

Passages: PAPER.md:114 (Eq. 12), :128 (Eq. 15), :136 (Eq. 16), :159 (Eq. 17), :170 (Eq. 19),
:176-182 (seeds, flags, continuation), :463-471 (App. C).
"""
import os

import numpy as np
import pytest

from paper_2506_02121_b200.configs import CONFIGS

HERE = os.path.dirname(os.path.abspath(__file__))


def cplx(a):
    return a[..., 0] + 1j * a[..., 1]


def c_phi(kappa_s, gamma, phi):
    return (1.0 - kappa_s) * np.exp(-1j * phi) - gamma


def match_sets(a, b):
    """Greedy-free check: sort-free nearest neighbour, returns (max distance, bijective)."""
    d = np.abs(a[:, None] - b[None, :])
    j = d.argmin(axis=1)
    return d[np.arange(len(a)), j].max(), len(set(j.tolist())) == len(b)


# ---------------------------------------------------------------------------------------------
# P1  Einstein ring: one unit star, kappa_s = gamma = 0  ->  z^2 = e^{i phi}, caustic = 0
# ---------------------------------------------------------------------------------------------
def test_p1_einstein_ring(orc):
    z0 = 0.37 - 0.21j  # translation invariance; also keeps seeds off the symmetric real axis
    xy = np.array([[z0.real, z0.imag]])
    m = np.array([1.0])
    num_phi = 64
    roots, iters, unconv = orc.critical_curves(xy, m, 0.0, 0.0, num_phi)
    assert unconv.sum() == 0
    z = cplx(roots) - z0
    phi = 2 * np.pi * np.arange(num_phi) / num_phi
    assert np.abs(np.abs(z) - 1.0).max() < 1e-15 * 4
    for j in range(num_phi):
        want = np.array([np.exp(0.5j * phi[j]), -np.exp(0.5j * phi[j])])
        err, bij = match_sets(z[j], want)
        assert bij and err < 4e-15
    w = cplx(orc.caustics(xy, m, 0.0, 0.0, roots))
    assert np.abs(w - z0).max() < 4e-15  # point caustic at the star (lens map of the ring)


# ---------------------------------------------------------------------------------------------
# P2  Chang–Refsdal: one star of mass m with shear and smooth matter -> z^2 = m / c(phi)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kappa_s,gamma,mass", [(0.2, 0.35, 1.0), (0.0, 0.3, 2.5), (0.1, 0.1, 0.3)])
def test_p2_chang_refsdal_roots(orc, kappa_s, gamma, mass):
    z0 = -1.3 + 0.8j
    xy = np.array([[z0.real, z0.imag]])
    m = np.array([mass])
    num_phi = 200
    roots, iters, unconv = orc.critical_curves(xy, m, kappa_s, gamma, num_phi)
    assert unconv.sum() == 0
    z = cplx(roots) - z0
    phi = 2 * np.pi * np.arange(num_phi) / num_phi
    for j in range(num_phi):
        r = np.sqrt(mass / c_phi(kappa_s, gamma, phi[j]))
        err, bij = match_sets(z[j], np.array([r, -r]))
        assert bij and err < 1e-14, (j, err)
    # caustic of the closed-form critical point through Eq. 12 written out for one star
    w = cplx(orc.caustics(xy, m, kappa_s, gamma, roots))
    zz = cplx(roots)
    want = (1 - kappa_s) * zz + gamma * np.conj(zz) - mass / (np.conj(zz) - np.conj(z0))
    assert np.abs(w - want).max() < 1e-14


def test_p2_chang_refsdal_cusps_golden(orc):
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "chang_refsdal_cusps.txt"))
            if not l.startswith("#")]
    for ks, g, re_cusp, im_cusp in rows:
        ks, g, re_cusp, im_cusp = float(ks), float(g), float(re_cusp), float(im_cusp)
        xy = np.array([[0.0, 0.0]])
        m = np.array([1.0])
        num_phi = 400  # even: row 0 is phi = 0, row 200 is phi = pi
        roots, _, unconv = orc.critical_curves(xy, m, ks, g, num_phi)
        assert unconv.sum() == 0
        w = cplx(orc.caustics(xy, m, ks, g, roots))
        w0 = np.sort_complex(w[0])
        assert abs(w0[0] + re_cusp) < 1e-14 and abs(w0[1] - re_cusp) < 1e-14
        wpi = w[num_phi // 2]
        assert np.abs(wpi.real).max() < 1e-14
        assert np.abs(np.sort(wpi.imag) - np.array([-im_cusp, im_cusp])).max() < 1e-14


# ---------------------------------------------------------------------------------------------
# P3  Equal-mass binary without shear: u = z^2 solves a quadratic
#     e^{-i phi} u^2 - (2 b^2 e^{-i phi} + 2 m) u + (b^4 e^{-i phi} - 2 m b^2) = 0, stars at +-b
# ---------------------------------------------------------------------------------------------
def test_p3_equal_mass_binary(orc):
    b = 0.8 * np.exp(0.3j)
    mass = 0.7
    xy = np.array([[b.real, b.imag], [-b.real, -b.imag]])
    m = np.array([mass, mass])
    num_phi = 90
    roots, _, unconv = orc.critical_curves(xy, m, 0.0, 0.0, num_phi)
    assert unconv.sum() == 0
    z = cplx(roots)
    for j in range(num_phi):
        e = np.exp(-2j * np.pi * j / num_phi)
        u = np.roots([e, -(2 * b * b * e + 2 * mass), b ** 4 * e - 2 * mass * b * b])
        want = np.concatenate([np.sqrt(u), -np.sqrt(u)])
        err, bij = match_sets(z[j], want)
        assert bij and err < 1e-13, (j, err)


# ---------------------------------------------------------------------------------------------
# P4  Companion matrix: expand P(z) = F(z) prod (z - z_i)^2 (Eq. 16) and take np.roots
# ---------------------------------------------------------------------------------------------
def expanded_polynomial(zs, ms, kappa_s, gamma, phi):
    """-c(phi) prod_i (z-z_i)^2 + sum_i m_i prod_{j != i} (z-z_j)^2, highest power first."""
    N = len(zs)
    full = np.array([1.0 + 0j])
    for zi in zs:
        full = np.polymul(full, np.polymul([1, -zi], [1, -zi]))
    p = -c_phi(kappa_s, gamma, phi) * full
    for i in range(N):
        part = np.array([1.0 + 0j])
        for jj in range(N):
            if jj != i:
                part = np.polymul(part, np.polymul([1, -zs[jj]], [1, -zs[jj]]))
        p = np.polyadd(p, ms[i] * part)
    return p


@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 6])
def test_p4_companion_matrix(orc, N):
    rng = np.random.default_rng(100 + N)
    zs = (rng.uniform(-2, 2, N) + 1j * rng.uniform(-2, 2, N))
    ms = rng.uniform(0.3, 2.0, N)
    kappa_s, gamma = 0.15, 0.3
    xy = np.stack([zs.real, zs.imag], axis=1)
    num_phi = 24
    roots, _, unconv = orc.critical_curves(xy, ms, kappa_s, gamma, num_phi)
    assert unconv.sum() == 0
    z = cplx(roots)
    assert z.shape == (num_phi, 2 * N)
    for j in range(num_phi):
        p = expanded_polynomial(zs, ms, kappa_s, gamma, 2 * np.pi * j / num_phi)
        assert len(p) == 2 * N + 1  # degree exactly 2N
        err, bij = match_sets(z[j], np.roots(p))
        assert bij and err < 1e-8, (N, j, err)


# ---------------------------------------------------------------------------------------------
# P5-P7  invariants on the synthetic workloads: Vieta sums, det J, long-double Newton residual
# ---------------------------------------------------------------------------------------------
def _field(orc, cfg):
    return orc.star_field(cfg.seed, cfg.N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)


def check_row_invariants(orc, xy, m, kappa_s, gamma, row_index, num_phi, z, min_sep=1e-6):
    """All pins that hold for ANY claimed root set of one phase (also used by the GPU tests)."""
    zs = xy[:, 0] + 1j * xy[:, 1]
    N = len(m)
    assert z.shape == (2 * N,)
    phi = 2 * np.pi * row_index / num_phi
    c = c_phi(kappa_s, gamma, phi)
    # Vieta: sum z_k = 2 sum z_i ; sum z_k^2 = 2 sum z_i^2 + 2 (sum m_i)/c(phi)
    s1, s2 = z.sum(), (z * z).sum()
    assert abs(s1 - 2 * zs.sum()) <= 1e-12 * np.abs(z).sum()
    assert abs(s2 - (2 * (zs * zs).sum() + 2 * m.sum() / c)) <= 1e-12 * (np.abs(z) ** 2).sum()
    res = orc.residuals(xy, m, kappa_s, gamma, row_index, num_phi,
                        np.stack([z.real, z.imag], axis=1), long_double=True)
    ulp = np.spacing(np.abs(z))
    # residual certificate: the long-double Newton step from the fp64 root is at rounding level.  "Rounding level" is
    # the spacing of z, or -- for an ill-conditioned root (small |F'|) -- what the fp64 evaluation of F itself allows:
    # F is a sum of N terms m_i/(z-z_i)^2 added one after the other, every addition rounding by up to
    # 2^-53 |partial sum| <= 2^-53 sum |terms|; N independent roundings add up like a random walk, so F carries
    # |dF| ~ sqrt(N) 2^-53 sum |terms| and the iteration cannot place the root better than |dF|/|F'| (DESIGN.md reading
    # R16; the outer pair of cfg4 near phi = 0 sits at |z| ~ 2R where every term has the same phase and |F'| ~ 2e-4).
    # The factor 4 is the margin over that estimate; `test_r16_condition_term_on_the_oracles_own_cfg4_rows` shows the
    # oracle's own double solve needs the term on those rows and its long-double solve does not.
    plain = 4 * ulp + 1e-13
    over = np.where(res["newton"] > plain)[0]          # only these need the conditioning term (few, if any)
    for k in over:
        floor = 4 * np.sqrt(N) * 2.0 ** -53 * (m / np.abs(z[k] - zs) ** 2).sum() / np.abs(res["Fp"][k])
        assert res["newton"][k] <= plain[k] + floor, (k, res["newton"][k], plain[k], floor)
    assert len(over) <= max(2, len(z) // 1000)
    res["needed_condition_term"] = over
    # scaled det J bound (App. C linearised)
    bound = 1e-10 + 4 * (1 - kappa_s) * np.abs(res["Fp"]) * 2.0 ** -52 * (1 + np.abs(z))
    assert np.all(np.abs(res["inv_mu"]) <= bound), (np.abs(res["inv_mu"]) / bound).max()
    # distinct roots
    order = np.argsort(z.real)
    zr = z[order]
    sep = np.inf
    for sh in range(1, 8):
        sep = min(sep, np.abs(zr[sh:] - zr[:-sh]).min()) if len(zr) > sh else sep
    assert sep > min_sep
    return res


@pytest.mark.parametrize("name,nrows", [("cfg1", 1000), ("cfg2", 40)])
def test_p5_p6_p7_invariants_full_chain(orc, name, nrows):
    cfg = CONFIGS[name]
    xy, m, R = _field(orc, cfg)
    roots, iters, unconv = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, cfg.num_phi,
                                                   np.arange(nrows), cfg.tol, cfg.max_iter)
    assert unconv.sum() == 0 and iters.max() < cfg.max_iter
    z = cplx(roots)
    for j in range(0, nrows, max(1, nrows // 25)):
        res = check_row_invariants(orc, xy, m, cfg.kappa_s, cfg.gamma, j, cfg.num_phi, z[j])
        if name in ("cfg1", "cfg2"):
            assert np.abs(res["inv_mu"]).max() <= 1e-10  # the plain BASELINE.json invariant


def test_p5_p6_p7_invariants_cfg3_row(orc):
    cfg = CONFIGS["cfg3"]
    xy, m, R = _field(orc, cfg)
    rows = [0, 1, 2]
    roots, iters, unconv = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, cfg.num_phi,
                                                   rows, cfg.tol, cfg.max_iter)
    assert unconv.sum() == 0
    for q, j in enumerate(rows):
        check_row_invariants(orc, xy, m, cfg.kappa_s, cfg.gamma, j, cfg.num_phi, cplx(roots)[q])


def test_r16_condition_term_on_the_oracles_own_cfg4_rows(orc):
    """DESIGN.md reading R16 on the ORACLE's rows (no GPU): the conditioning term of the residual certificate is what
    an fp64 solve needs, not a kernel allowance.  cfg4, row 0 (phi = 0: |c(phi)| = 0.05, the outer pair at |z| ~ 2R,
    PAPER.md:422 fn. 7, with |F'| ~ 2e-4) and row 5000 (phi = pi, no such pair): the double solve passes every row
    invariant, needs the term for a handful of roots on row 0 and for none on row 5000; the long-double solve of the
    same rows, rounded to fp64, needs it nowhere."""
    cfg = CONFIGS["cfg4"]
    xy, m, R = _field(orc, cfg)
    rows = [0, 5000]
    need = {}
    for ld in (False, True):
        roots, iters, unconv = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, cfg.num_phi, rows, cfg.tol,
                                                       cfg.max_iter, long_double=ld)
        assert unconv.sum() == 0 and iters.max() < cfg.max_iter
        for q, j in enumerate(rows):
            res = check_row_invariants(orc, xy, m, cfg.kappa_s, cfg.gamma, j, cfg.num_phi, cplx(roots)[q])
            need[(ld, j)] = np.abs(cplx(roots)[q][res["needed_condition_term"]])   # |z| of the roots that needed it
    assert 1 <= len(need[(False, 0)]) <= 20          # the fp64 floor is real: the oracle's own double row needs it
    assert np.all(need[(False, 0)] > 1.5 * R)        # ... and only for the outer pair
    assert len(need[(False, 5000)]) == 0
    assert len(need[(True, 0)]) == 0 and len(need[(True, 5000)]) == 0


def test_double_vs_long_double_rows(orc):
    cfg = CONFIGS["cfg2"]
    xy, m, R = _field(orc, cfg)
    rows = [0, 1, 2000, 3999]
    rd, _, _ = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, cfg.num_phi, rows)
    rl, _, _ = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, cfg.num_phi, rows, long_double=True)
    for q in range(len(rows)):
        err, bij = match_sets(cplx(rd)[q], cplx(rl)[q])
        assert bij and err < 1e-12


def test_seed_independence(orc):
    """The result is the root SET: a different seeding path reaches the same set."""
    cfg = CONFIGS["cfg1"]
    xy, m, R = _field(orc, cfg)
    a, _, _ = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, cfg.num_phi, [500])
    b, _, _ = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, cfg.num_phi, np.arange(501))
    err, bij = match_sets(cplx(a)[0], cplx(b)[500])
    assert bij and err < 1e-13


# ---------------------------------------------------------------------------------------------
# P8  continuity in phi: z_k(phi + dphi) - z_k(phi) = z'_k dphi + O(dphi^2),
#     z' = -i (1-kappa_s) e^{-i phi} / F'(z)   (from dF = 0)
# ---------------------------------------------------------------------------------------------
def test_p8_continuity(orc):
    cfg = CONFIGS["cfg2"]
    xy, m, R = _field(orc, cfg)
    nrows = 12
    roots, _, unconv = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, cfg.num_phi,
                                               np.arange(nrows))
    z = cplx(roots)
    dphi = 2 * np.pi / cfg.num_phi
    zp = []
    for j in range(nrows):
        res = orc.residuals(xy, m, cfg.kappa_s, cfg.gamma, j, cfg.num_phi, roots[j])
        zp.append(-1j * (1 - cfg.kappa_s) * np.exp(-1j * j * dphi) / res["Fp"])
    for j in range(nrows - 1):
        # column k of row j+1 continues column k of row j:
        # trapezoid rule on z' leaves O(dphi^3); the Euler step leaves O(dphi^2)
        step = z[j + 1] - z[j]
        trap = 0.5 * (zp[j] + zp[j + 1]) * dphi
        assert np.abs(step - trap).max() < 1e-3 * np.abs(step).max()
        assert np.abs(step - zp[j] * dphi).max() < 0.02 * np.abs(step).max()
        assert np.abs(step).max() < 0.05


# ---------------------------------------------------------------------------------------------
# P9  outer pair: far from the field the lens is Chang–Refsdal with the total mass
#     (PAPER.md:422 fn. 7): if kappa_star > |c(phi)| two roots sit near |z| = R sqrt(kappa_star/|c|)
# ---------------------------------------------------------------------------------------------
def test_p9_outer_pair(orc):
    cfg = CONFIGS["cfg4"]
    N = 600
    xy, m, R = orc.star_field(3, N, cfg.kappa_star, cfg.mass_model, cfg.mass_params)
    rows = [0]
    roots, _, unconv = orc.critical_curve_rows(xy, m, cfg.kappa_s, cfg.gamma, 1000, rows)
    assert unconv.sum() == 0
    z = cplx(roots)[0]
    c = abs(c_phi(cfg.kappa_s, cfg.gamma, 0.0))
    assert cfg.kappa_star > c
    want = R * np.sqrt(cfg.kappa_star / c)
    outer = np.sort(np.abs(z))[-2:]
    assert np.all(np.abs(outer / want - 1) < 0.03), (outer, want)
    assert np.sort(np.abs(z))[-3] < 1.2 * R


# ---------------------------------------------------------------------------------------------
# orientation: stars lie in negative-parity regions
# ---------------------------------------------------------------------------------------------
def test_parity_sign_near_stars(orc):
    cfg = CONFIGS["cfg1"]
    xy, m, R = _field(orc, cfg)
    pts = xy + np.array([1e-3, 0.0])
    res = orc.residuals(xy, m, cfg.kappa_s, cfg.gamma, 0, 1, pts)
    assert np.all(res["inv_mu"] < 0)


# ---------------------------------------------------------------------------------------------
# root-set matching against scipy's assignment solver
# ---------------------------------------------------------------------------------------------
def test_match_root_sets_vs_assignment(orc):
    from scipy.optimize import linear_sum_assignment
    rng = np.random.default_rng(7)
    S, n = 6, 40
    b = rng.normal(size=(S, n, 2)) * 10
    a = np.empty_like(b)
    for s in range(S):
        a[s] = b[s][rng.permutation(n)] + rng.normal(size=(n, 2)) * 1e-12
    a[4, 3] = a[4, 5]          # duplicate: not a bijection
    a[5, 0, 0] += 1e-3         # one root off by more than the tolerance
    err, bij = orc.match_root_sets(a, b, 1e-10)
    assert bij.tolist() == [1, 1, 1, 1, 0, 0]
    for s in range(4):
        d = np.linalg.norm(a[s][:, None, :] - b[s][None, :, :], axis=2)
        r, c = linear_sum_assignment(d)
        assert abs(d[r, c].max() - err[s]) < 1e-18 + 1e-6 * err[s]
    assert abs(err[5] - 1e-3) < 1e-9


# ---------------------------------------------------------------------------------------------
# star-field generator: Philox known answers, geometry, statistics, analytic mass CDFs
# ---------------------------------------------------------------------------------------------
def test_philox_known_answers(orc):
    for line in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")):
        if line.startswith("#"):
            continue
        w = [int(x, 16) for x in line.split()]
        assert orc.philox4x32_10(w[0:4], w[4:6]) == w[6:10]


def test_star_field_geometry_and_stats(orc):
    from scipy import stats
    N = 20000
    xy, m, R = orc.star_field(0, N, 0.2, 0)
    assert R == np.sqrt(N / 0.2)
    r2 = (xy ** 2).sum(axis=1) / R ** 2
    assert r2.max() < 1.0
    assert np.all(m == 1.0)
    assert stats.kstest(r2, "uniform").pvalue > 1e-3          # uniform in area
    ang = (np.arctan2(xy[:, 1], xy[:, 0]) + np.pi) / (2 * np.pi)
    assert stats.kstest(ang, "uniform").pvalue > 1e-3
    assert abs(r2.mean() - 0.5) < 0.01                         # <|z|^2> = R^2/2
    # different seeds, same seed
    xy2, _, _ = orc.star_field(1, N, 0.2, 0)
    xy3, _, _ = orc.star_field(0, N, 0.2, 0)
    assert np.array_equal(xy, xy3) and not np.array_equal(xy, xy2)
    # prefix property of a counter-based generator: star i does not depend on N (up to the R scale)
    xy4, _, R4 = orc.star_field(0, 100, 0.2, 0)
    assert np.allclose(xy4 / R4, xy[:100] / R, rtol=0, atol=1e-15)


def _broken_power_law_cdf(mgrid, p):
    """Forward CDF by direct numerical integration of the continuous broken power law."""
    m0, m1, m2, m3, a1, a2, a3 = p
    A2 = m1 ** (a2 - a1)
    A3 = A2 * m2 ** (a3 - a2)

    def pdf(x):
        return np.where(x < m1, x ** -a1, np.where(x < m2, A2 * x ** -a2, A3 * x ** -a3))
    xs = np.exp(np.linspace(np.log(m0), np.log(m3), 400001))
    f = pdf(xs)
    cum = np.concatenate([[0], np.cumsum(0.5 * (f[1:] + f[:-1]) * np.diff(xs))])
    cum /= cum[-1]
    return np.interp(mgrid, xs, cum)


def test_rectangular_star_field_geometry_and_stats(orc):
    """Stars of Section 4.2's rectangular field: Eq. 9 with A_star = 4 c1 c2 and
    sum m = N gives the corner; x/c1 and y/c2 are independent and uniform on [-1, 1); the stars the disk recipe
    accepts at its first attempt are the same points of the unit square."""
    from scipy import stats
    N, kstar, aspect = 20000, 0.35, 1.7
    xy, m, c1, c2 = orc.star_field_rect(3, N, kstar, aspect, 1)
    assert abs(c1 / c2 - aspect) < 1e-14 and abs(np.pi * m.sum() / (4 * c1 * c2) - kstar) < 1e-12   # Eq. 9
    assert abs(m.sum() - N) < 1e-9 * N
    u, v = xy[:, 0] / c1, xy[:, 1] / c2
    assert np.abs(u).max() < 1 and np.abs(v).max() < 1 and np.abs(u).max() > 0.999
    assert stats.kstest((u + 1) / 2, "uniform").pvalue > 1e-3 and stats.kstest((v + 1) / 2, "uniform").pvalue > 1e-3
    assert abs(np.corrcoef(u, v)[0, 1]) < 0.03
    occupancy = np.histogram2d(u, v, bins=8, range=[[-1, 1], [-1, 1]])[0]
    assert stats.chisquare(occupancy.ravel()).pvalue > 1e-3                       # uniform in area
    # same seed -> same masses as the disk field; first-attempt stars of the disk are the same unit-square points
    dxy, dm, R = orc.star_field(3, N, kstar, 1)
    assert np.array_equal(dm, m)
    first = u ** 2 + v ** 2 < 1 - 1e-12
    assert 0.75 < first.mean() < 0.82                                             # pi/4
    assert np.abs(dxy[first, 0] / R - u[first]).max() < 1e-15 and np.abs(dxy[first, 1] / R - v[first]).max() < 1e-15
    xy2, _, _, _ = orc.star_field_rect(4, N, kstar, aspect, 1)
    assert not np.array_equal(xy, xy2)
    with pytest.raises(RuntimeError):
        orc.star_field_rect(0, 10, 0.4, 0.0)


def test_star_field_mass_functions(orc):
    from scipy import stats
    N = 40000
    # Salpeter
    xy, m, R = orc.star_field(0, N, 0.45, 1)
    assert abs(m.mean() - 1) < 1e-12 and abs(m.sum() - N) < 1e-8
    assert abs(m.max() / m.min()) <= 1.0 / 0.08 + 1e-9
    raw = m / m.min() * 0.08 if False else None  # (scale unknown after normalisation; use ratios)
    lo, hi, al = 0.08, 1.0, 2.35
    scale = None
    # recover the scale: unnormalised mean of the power law
    e1, e2 = 1 - al, 2 - al
    mean_raw = ((hi ** e2 - lo ** e2) / e2) / ((hi ** e1 - lo ** e1) / e1)
    raw = m * mean_raw  # approximately the unnormalised masses (sample mean ~ population mean)
    cdf = lambda x: np.clip((x ** e1 - lo ** e1) / (hi ** e1 - lo ** e1), 0, 1)
    assert stats.kstest(raw, cdf).pvalue > 1e-4
    # Kroupa-like broken power law
    p = (0.01, 0.08, 0.5, 1.5, 0.3, 1.3, 2.3)
    xy, m, R = orc.star_field(0, N, 0.2, 2)
    assert abs(m.mean() - 1) < 1e-12
    assert m.max() / m.min() <= 150.0 + 1e-6
    xs = np.exp(np.linspace(np.log(p[0]), np.log(p[3]), 200001))
    cdfx = _broken_power_law_cdf(xs, p)
    pdf_mean = np.trapezoid(xs * np.gradient(cdfx, xs), xs)
    raw = m * pdf_mean
    assert stats.kstest(raw, lambda x: np.interp(x, xs, cdfx)).pvalue > 1e-4
    # explicit parameters == defaults
    xy2, m2, _ = orc.star_field(0, N, 0.2, 2, p)
    assert np.array_equal(m, m2) and np.array_equal(xy, xy2)


def test_star_sums_regular_polygon_closed_form(orc):
    """K equal stars of mass m on the circle |z| = a at the K-th roots of a^K (textbook partial fractions):
    sum_j 1/(z - a w^j) = K z^(K-1)/(z^K - a^K) =: g(z), so S1 = g, Sm = m g, S2 = -m g', S3 = m g''/2.
    Pins every sum the oracle's star loop forms (power, sign, mass factor), also for points inside the ring."""
    K, a, mass = 7, 1.7, 0.6
    zs = a * np.exp(2j * np.pi * np.arange(K) / K)
    xy = np.stack([zs.real, zs.imag], axis=1)
    m = np.full(K, mass)
    pts = np.array([[0.3, -0.2], [2.5, 1.1], [-4.0, 0.7], [0.0, 3.3], [1.0, 1.0]])
    z = pts[:, 0] + 1j * pts[:, 1]
    q = z ** K - a ** K
    g = K * z ** (K - 1) / q
    g1 = K * (K - 1) * z ** (K - 2) / q - (K * z ** (K - 1)) ** 2 / q ** 2
    g2 = (K * (K - 1) * (K - 2) * z ** (K - 3) / q - 3 * K * (K - 1) * z ** (K - 2) * K * z ** (K - 1) / q ** 2
          + 2 * (K * z ** (K - 1)) ** 3 / q ** 3)
    for ld in (False, True):
        out = orc.star_sums(xy, m, pts, long_double=ld)
        S1, S2, S3, Sm = (out[:, 0] + 1j * out[:, 1], out[:, 2] + 1j * out[:, 3], out[:, 4] + 1j * out[:, 5],
                          out[:, 6] + 1j * out[:, 7])
        assert np.abs(S1 - g).max() < 1e-13
        assert np.abs(Sm - mass * g).max() < 1e-13
        assert np.abs(S2 + mass * g1).max() < 1e-12
        assert np.abs(S3 - mass * g2 / 2).max() < 1e-12


def test_star_sums_consistent_with_residuals_and_caustics(orc):
    """F = gamma + S2 - (1-kappa_s) e^{-i phi}, F' = -2 S3 (Eq. 15, 19) and w = (1-kappa_s) z + gamma conj z - conj Sm
    (Eq. 12): the exported sums are the ones the solver and the caustic map use."""
    xy, m, R = orc.star_field(3, 300, 0.3, 2)
    pts = np.random.default_rng(0).normal(size=(50, 2)) * R * 0.6
    ks, g = 0.15, 0.35
    out = orc.star_sums(xy, m, pts)
    res = orc.residuals(xy, m, ks, g, 7, 64, pts)
    phi = 2 * np.pi * 7 / 64
    F = g + (out[:, 2] + 1j * out[:, 3]) - (1 - ks) * np.exp(-1j * phi)
    assert np.abs(F - res["F"]).max() < 1e-13 * (1 + np.abs(F).max())
    assert np.abs(-2 * (out[:, 4] + 1j * out[:, 5]) - res["Fp"]).max() < 1e-13 * (1 + np.abs(res["Fp"]).max())
    w = cplx(orc.caustics(xy, m, ks, g, pts, long_double=True))
    z = pts[:, 0] + 1j * pts[:, 1]
    assert np.abs((1 - ks) * z + g * np.conj(z) - np.conj(out[:, 6] + 1j * out[:, 7]) - w).max() < 1e-12


def test_vieta_residuals_certify_complete_root_sets(orc):
    """orc_vieta_residuals against things it does not compute itself: roots of the EXPANDED polynomial from numpy's
    companion-matrix solver (N <= 5) must pass; the closed-form Chang-Refsdal roots must pass; and a set with one
    root replaced by a copy of another fails by exactly the displacement |z_b - z_a| / sum |z_k|."""
    rng = np.random.default_rng(21)
    for N in (1, 2, 3, 5):
        zs = rng.uniform(-2, 2, N) + 1j * rng.uniform(-2, 2, N)
        ms = rng.uniform(0.3, 1.5, N)
        xy = np.stack([zs.real, zs.imag], axis=1)
        kappa_s, gamma, num_phi = 0.15, 0.3, 7
        rows = []
        for j in range(num_phi):
            r = np.roots(expanded_polynomial(zs, ms, kappa_s, gamma, 2 * np.pi * j / num_phi))
            assert len(r) == 2 * N
            rows.append(np.stack([r.real, r.imag], axis=1))
        rows = np.stack(rows)
        e1, e2 = orc.vieta_residuals(xy, ms, kappa_s, gamma, rows)
        assert e1.max() < 1e-9 and e2.max() < 1e-9            # numpy's roots of an expanded polynomial: ~1e-11
        # a sub-grid of a finer one: rows 3..4 of 14 phases are phases 2 pi 3/14, 2 pi 4/14
        fine = np.stack([np.stack([r.real, r.imag], axis=1) for r in
                         (np.roots(expanded_polynomial(zs, ms, kappa_s, gamma, 2 * np.pi * j / 14)) for j in (3, 4))])
        f1, f2 = orc.vieta_residuals(xy, ms, kappa_s, gamma, fine, j_offset=3, num_phi_total=14)
        assert f1.max() < 1e-9 and f2.max() < 1e-9
        w1, w2 = orc.vieta_residuals(xy, ms, kappa_s, gamma, fine, j_offset=0, num_phi_total=14)
        assert w2.max() > 1e-4                                  # the wrong phase: the second sum notices
        if N >= 2:
            bad = rows.copy()
            bad[2, 0] = bad[2, 1]                                # one root duplicated, one missing
            b1, b2 = orc.vieta_residuals(xy, ms, kappa_s, gamma, bad)
            shift = abs(cplx(rows[2, 1]) - cplx(rows[2, 0]))
            assert abs(b1[2] - shift / np.abs(cplx(bad[2])).sum()) < 1e-9 and b1[2] > 1e-3
            assert np.delete(b1, 2).max() < 1e-9
    # Chang-Refsdal closed form z = +-sqrt(m / c(phi))
    m, kappa_s, gamma, num_phi = 0.8, 0.2, 0.35, 12
    rows = []
    for j in range(num_phi):
        z = np.sqrt(m / c_phi(kappa_s, gamma, 2 * np.pi * j / num_phi))
        rows.append([[z.real, z.imag], [-z.real, -z.imag]])
    e1, e2 = orc.vieta_residuals(np.zeros((1, 2)), np.array([m]), kappa_s, gamma, np.array(rows))
    assert e1.max() < 1e-15 and e2.max() < 1e-15
