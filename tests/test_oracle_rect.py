"""Pins of the oracle's rectangular-sheet formulas (Appendix A-B, Eq. B2, B7, B9) and of its solver with
the extra t - 1 roots, against things other than the formulas themselves: the deflection of a uniform rectangle from
potential theory (a boundary integral), finite differences, and companion-matrix roots of the expanded polynomial."""
import numpy as np
import pytest
from scipy import integrate

from test_oracle_pins import cplx, match_sets


def rectangle_deflection(kappa_star, c1, c2, p):
    """Deflection of a uniform sheet of convergence kappa_star on [-c1,c1] x [-c2,c2] at the inside point p:
    alpha = (kappa/pi) int (p - r')/|p - r'|^2 dA' = -(kappa/pi) oint ln|p - r'| n dl (Green), n the outward normal.
    Four smooth 1-D integrals."""
    px, py = p.real, p.imag

    def edge(f, a, b):
        return integrate.quad(f, a, b, epsabs=1e-13, epsrel=1e-13, limit=200)[0]

    right = edge(lambda y: 0.5 * np.log((px - c1) ** 2 + (py - y) ** 2), -c2, c2)      # n = +x
    left = edge(lambda y: 0.5 * np.log((px + c1) ** 2 + (py - y) ** 2), -c2, c2)       # n = -x
    top = edge(lambda x: 0.5 * np.log((px - x) ** 2 + (py - c2) ** 2), -c1, c1)        # n = +y
    bottom = edge(lambda x: 0.5 * np.log((px - x) ** 2 + (py + c2) ** 2), -c1, c1)     # n = -y
    return -(kappa_star / np.pi) * ((right - left) + 1j * (top - bottom))


@pytest.mark.parametrize("c1,c2", [(3.0, 3.0), (5.0, 2.0), (1.5, 4.0)])
def test_b2_is_minus_the_deflection_of_the_uniform_rectangle(orc, c1, c2):
    """alpha_s compensates the stars' mean deflection: alpha_s = -(deflection of the sheet) inside the rectangle
    (as -kappa_star z does for the disc, Eq. A1), up to the truncation bound B4."""
    ks = 0.37
    c = abs(c1 + 1j * c2)
    pts = np.array([[0.0, 0.0], [0.4, -0.3], [-1.0, 0.9], [0.9 * min(c1, c2), 0.1], [-0.2, -0.8 * min(c1, c2)]])
    t = 201
    a, _, _ = orc.rect_sheet(ks, c1, c2, t, pts)
    for z, got in zip(pts[:, 0] + 1j * pts[:, 1], a):
        want = -rectangle_deflection(ks, c1, c2, z)
        bound = ks / np.pi * 4 / (t + 1) * (abs(z) / c) ** (t + 1) * (c + abs(z)) / (1 - abs(z) / c)
        assert abs(got - want) < 1e-10 + bound, (z, got, want)
    assert abs(a[0]) < 1e-13                      # alpha_s(0) = 0 by symmetry


def test_b4_bounds_the_truncation_error(orc):
    ks, c1, c2 = 0.4, 4.0, 2.5
    c = abs(c1 + 1j * c2)
    rng = np.random.default_rng(0)
    pts = rng.uniform(-1, 1, size=(40, 2)) * np.array([c1, c2]) * 0.8
    exact, _, _ = orc.rect_sheet(ks, c1, c2, 801, pts)
    z = np.abs(pts[:, 0] + 1j * pts[:, 1])
    for t in (5, 11, 21, 41):
        a, _, _ = orc.rect_sheet(ks, c1, c2, t, pts)
        bound = ks / np.pi * 4 / (t + 1) * (z / c) ** (t + 1) * (c + z) / (1 - z / c)
        assert (np.abs(a - exact) <= bound + 1e-13).all()
    assert orc.rect_truncation(ks, c1, c2, 1.5, 1e-9) % 2 == 1
    t = orc.rect_truncation(ks, c1, c2, 1.5, 1e-9)
    s = 1.5
    assert ks / np.pi * 4 / (t + 1) * s ** -(t + 1) * c * (s + 1) / (s - 1) <= 1e-9
    r = ((t - 1) * np.arctan2(c2, c1)) % np.pi
    assert 0.1 * np.pi <= r <= 0.9 * np.pi


@pytest.mark.parametrize("ks,c1,c2,s,eps", [(0.4, 4.0, 2.5, 1.5, 1e-9), (0.3, 3.0, 3.0, 1.2, 1e-6), (0.2, 10.0, 1.0, 2.0, 1e-12),
                                             (0.45, 5.0, 5.0 * np.tan(np.pi / 10), 1.5, 1e-9), (0.1, 1.0, 2.0, 1.05, 1e-3)])
def test_truncation_power_is_the_smallest_admissible_one(orc, ks, c1, c2, s, eps):
    """`orc_rect_truncation` returns THE SMALLEST odd t that meets both rules of Appendix B: the error bound B5
     below eps on |z| <= |c|/s, and (t-1) Arg c at least 0.1 pi away from the multiples of pi
    (PAPER.md:456).  Brute force over every smaller odd power: each one breaks B5 or the Arg rule."""
    c, theta = abs(c1 + 1j * c2), np.arctan2(c2, c1)

    def b5_ok(t):
        return ks / np.pi * 4 / (t + 1) * s ** -(t + 1) * c * (s + 1) / (s - 1) <= eps

    def arg_ok(t):
        r = ((t - 1) * theta) % np.pi
        return 0.1 * np.pi <= r <= 0.9 * np.pi

    t = orc.rect_truncation(ks, c1, c2, s, eps)
    assert t % 2 == 1 and b5_ok(t) and arg_ok(t)
    smaller = [q for q in range(1, t, 2) if b5_ok(q) and arg_ok(q)]
    assert smaller == [], smaller
    # the cases cover both ways of stopping: B5 alone decides (t - 2 breaks it), or the Arg rule pushed t up
    if b5_ok(t - 2):
        assert not arg_ok(t - 2)


@pytest.mark.parametrize("t", [5, 9, 15])
def test_b7_b9_are_the_derivatives_of_b2(orc, t):
    """Wirtinger derivatives by central differences: d/dzbar = (d/dx + i d/dy)/2, d/dz = (d/dx - i d/dy)/2."""
    ks, c1, c2 = 0.3, 3.0, 2.0
    rng = np.random.default_rng(1)
    pts = rng.uniform(-1.5, 1.5, size=(12, 2))
    h = 1e-5

    def alpha(p):
        return orc.rect_sheet(ks, c1, c2, t, p)[0]

    def dzbar_of(f, p):
        dx = (f(p + [h, 0]) - f(p - [h, 0])) / (2 * h)
        dy = (f(p + [0, h]) - f(p - [0, h])) / (2 * h)
        return 0.5 * (dx + 1j * dy), 0.5 * (dx - 1j * dy)

    _, b7, b9 = orc.rect_sheet(ks, c1, c2, t, pts)
    d_zbar, d_z = dzbar_of(alpha, pts)
    assert np.abs(d_zbar - b7).max() < 1e-8
    assert np.abs(d_z - (-ks)).max() < 1e-8                     # B6
    d2, mixed = dzbar_of(lambda p: orc.rect_sheet(ks, c1, c2, t, p)[1], pts)
    assert np.abs(d2 - b9).max() < 1e-8 and np.abs(mixed).max() < 1e-8


def expanded_rect_polynomial(zs, ms, kappa_s, gamma, phi, kappa_star, c1, c2, t):
    """P(z) = F(z) prod (z - z_i)^2 with the sheet's polynomial written in real form: for odd t,
    conj(d alpha_s/d zbar) = kappa_star (1 - 4 theta/pi) - (4 kappa_star/pi) sum_{j = 2,4,..,t-1} sin(j theta)/j (z/|c|)^j,
    theta = Arg c  (reading R24; derived from B2, not copied from B7)."""
    theta, cabs = np.arctan2(c2, c1), np.hypot(c1, c2)
    G = np.zeros(t, complex)                                     # ascending powers 0 .. t-1
    G[0] = kappa_star * (1 - 4 * theta / np.pi)
    for j in range(2, t, 2):
        G[j] = -(4 * kappa_star / np.pi) * np.sin(j * theta) / j / cabs ** j
    coef = -G
    coef[0] += gamma - (1 - kappa_s) * np.exp(-1j * phi)
    const = np.poly1d(coef[::-1])
    prod = np.poly1d([1.0])
    for zi in zs:
        prod = prod * np.poly1d([1.0, -zi]) ** 2
    P = const * prod
    for i, (zi, mi) in enumerate(zip(zs, ms)):
        term = np.poly1d([mi])
        for j, zj in enumerate(zs):
            if j != i:
                term = term * np.poly1d([1.0, -zj]) ** 2
        P = P + term
    return P


@pytest.mark.parametrize("N,t", [(1, 3), (2, 5), (3, 5), (4, 7)])
def test_rect_solver_finds_all_2N_plus_t_minus_1_roots(orc, N, t):
    rng = np.random.default_rng(10 + N)
    c1, c2, ks_star = 3.0, 2.0, 0.4
    xy = rng.uniform(-1, 1, size=(N, 2)) * [c1 * 0.8, c2 * 0.8]
    m = rng.uniform(0.5, 1.5, size=N)
    kappa_s, gamma = 0.1, 0.25
    rows = np.array([1, 5, 11])
    roots, it, un = orc.rect_critical_curve_rows(xy, m, kappa_s, gamma, ks_star, c1, c2, t, 1.2 * np.hypot(c1, c2), 16, rows)
    assert un.sum() == 0 and roots.shape[1] == 2 * N + t - 1
    zs = xy[:, 0] + 1j * xy[:, 1]
    for q, j in enumerate(rows):
        P = expanded_rect_polynomial(zs, m, kappa_s, gamma, 2 * np.pi * j / 16, ks_star, c1, c2, t)
        assert P.order == 2 * N + t - 1
        want = np.roots(P.coeffs)
        err, bij = match_sets(cplx(roots[q]), want)
        assert bij and err < 1e-7 * (1 + np.abs(want).max()), err


def test_rect_caustics_follow_eq12_with_b2(orc):
    """w - [(1-kappa_s) z + gamma_eff zbar - conj(Sm + H(z))] = 0 with gamma_eff = gamma - kappa_star (1 - 4 theta/pi)
    and H(u) = -(4 kappa_star/pi) sum_{n odd, 3..t} sin((n-1) theta)/(n (n-1)) u^n/|c|^(n-1): the real-coefficient form
    the CUDA path uses (R24), here held against the oracle's literal B2."""
    rng = np.random.default_rng(3)
    c1, c2, kstar, t = 4.0, 2.5, 0.35, 9
    xy = rng.uniform(-1, 1, size=(6, 2)) * [c1, c2]
    m = rng.uniform(0.5, 1.5, size=6)
    pts = rng.uniform(-1, 1, size=(30, 2)) * [c1, c2]
    ks, g = 0.1, 0.2
    w = cplx(orc.rect_caustics(xy, m, ks, g, kstar, c1, c2, t, pts))
    z = pts[:, 0] + 1j * pts[:, 1]
    theta, cabs = np.arctan2(c2, c1), np.hypot(c1, c2)
    H = sum(-(4 * kstar / np.pi) * np.sin((n - 1) * theta) / (n * (n - 1)) * z ** n / cabs ** (n - 1) for n in range(3, t + 1, 2))
    sums = orc.star_sums(xy, m, pts)
    Sm = sums[:, 6] + 1j * sums[:, 7]
    want = (1 - ks) * z + (g - kstar * (1 - 4 * theta / np.pi)) * np.conj(z) - np.conj(Sm + H)
    assert np.abs(w - want).max() < 1e-12 * (1 + np.abs(want).max())
