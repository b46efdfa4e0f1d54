/* oracle/mlcc_oracle.c
 *
 * TEST INFRASTRUCTURE ONLY.  This is the plain, slow, CPU oracle for the hot path of
 * arXiv 2506.02121 (critical curves by Aberth–Ehrlich root finding, phase continuation,
 * caustic mapping, star-field generator, root-set matching).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 * The product (paper_2506_02121_b200/, include/) never imports, links or executes it,
 * and it shares no code, header, table or helper with the CUDA path.
 *
 * It is written from /root/reference/PAPER.md; every function cites the passage it follows
 * (PAPER.md:<line>).  Readings of silent / ambiguous passages are listed in DESIGN.md.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): Einstein ring, Chang–Refsdal closed form and
 * cusp positions, equal-mass binary closed form, companion-matrix eigenvalues (N <= 6),
 * Vieta sums, det J, long-double residual certificates, continuity in phi, outer root pair,
 * Philox known-answer vectors, generator statistics; closed loops by the binary-lens topologies and the
 * Einstein ring / Chang-Refsdal chain structure; distance maps by scipy's Euclidean distance transform,
 * a disc, and hand-worked rays (tests/test_oracle_loops_distance.py).
 * Parity unpinned: the mass functions and star positions "of the paper's fields" (the paper
 * publishes neither); both sides consume the same generated arrays.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fopenmp -fPIC -shared (oracle/build.py).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------------------------
 * double instantiation
 * ---------------------------------------------------------------------------------------- */
#define REAL double
#define CPLX double complex
#define NAME(x) x##_d
#define CREAL creal
#define CIMAG cimag
#define CABS cabs
#define CONJ conj
#define COS cos
#define SIN sin
#define PI_ 3.14159265358979323846264338327950288
#define CMPLX_(a, b) CMPLX((a), (b))
#include "aberth_generic.inc"
#undef REAL
#undef CPLX
#undef NAME
#undef CREAL
#undef CIMAG
#undef CABS
#undef CONJ
#undef COS
#undef SIN
#undef PI_
#undef CMPLX_

/* ------------------------------------------------------------------------------------------
 * long double instantiation
 * ---------------------------------------------------------------------------------------- */
#define REAL long double
#define CPLX long double complex
#define NAME(x) x##_ld
#define CREAL creall
#define CIMAG cimagl
#define CABS cabsl
#define CONJ conjl
#define COS cosl
#define SIN sinl
#define PI_ 3.14159265358979323846264338327950288L
#define CMPLX_(a, b) CMPLXL((a), (b))
#include "aberth_generic.inc"
#undef REAL
#undef CPLX
#undef NAME
#undef CREAL
#undef CIMAG
#undef CABS
#undef CONJ
#undef COS
#undef SIN
#undef PI_
#undef CMPLX_

/* ------------------------------------------------------------------------------------------
 * exported entry points (ctypes; complex numbers are interleaved (re, im) doubles)
 * ---------------------------------------------------------------------------------------- */

/* Sequential phase continuation over the whole grid:
 * row 0 from the cold seeds z_i +/- 1, row j+1 from row j.            */
int orc_critical_curves(const double *star_xy, const double *masses, int64_t N,
                        double kappa_s, double gamma, int64_t num_phi, double tol, int max_iter,
                        double *out_roots, int32_t *out_iters, int32_t *out_unconverged)
{
    if (N < 1 || num_phi < 1) return -2;
    int64_t *rows = (int64_t *)malloc(sizeof(int64_t) * (size_t)num_phi);
    if (!rows) return -1;
    for (int64_t j = 0; j < num_phi; ++j) rows[j] = j;
    int rc = curve_rows_d(star_xy, masses, N, kappa_s, gamma, num_phi, 0, rows, num_phi, tol,
                          max_iter, NULL, out_roots, out_iters, out_unconverged);
    free(rows);
    return rc;
}

/* Selected rows of the grid phi_j = 2 pi (j + j_offset)/num_phi_total, double arithmetic. */
int orc_critical_curve_rows(const double *star_xy, const double *masses, int64_t N,
                            double kappa_s, double gamma, int64_t num_phi_total, int64_t j_offset,
                            const int64_t *rows, int64_t nrows, double tol, int max_iter,
                            const double *init_roots, double *out_roots,
                            int32_t *out_iters, int32_t *out_unconverged)
{
    if (N < 1 || num_phi_total < 1 || nrows < 0) return -2;
    return curve_rows_d(star_xy, masses, N, kappa_s, gamma, num_phi_total, j_offset, rows, nrows,
                        tol, max_iter, init_roots, out_roots, out_iters, out_unconverged);
}

/* Same, long double arithmetic (results rounded to double on output). */
int orc_critical_curve_rows_ld(const double *star_xy, const double *masses, int64_t N,
                               double kappa_s, double gamma, int64_t num_phi_total, int64_t j_offset,
                               const int64_t *rows, int64_t nrows, double tol, int max_iter,
                               const double *init_roots, double *out_roots,
                               int32_t *out_iters, int32_t *out_unconverged)
{
    if (N < 1 || num_phi_total < 1 || nrows < 0) return -2;
    return curve_rows_ld(star_xy, masses, N, kappa_s, gamma, num_phi_total, j_offset, rows, nrows,
                         tol, max_iter, init_roots, out_roots, out_iters, out_unconverged);
}

int orc_caustics(const double *star_xy, const double *masses, int64_t N, double kappa_s,
                 double gamma, const double *points, int64_t P, double *out)
{
    if (N < 1 || P < 0) return -2;
    caustics_d(star_xy, masses, N, kappa_s, gamma, points, P, out);
    return 0;
}

int orc_caustics_ld(const double *star_xy, const double *masses, int64_t N, double kappa_s,
                    double gamma, const double *points, int64_t P, double *out)
{
    if (N < 1 || P < 0) return -2;
    caustics_ld(star_xy, masses, N, kappa_s, gamma, points, P, out);
    return 0;
}

/* F, F', 1/mu, |F|/|F'| at given points, long double (residual certificate). */
int orc_residuals_ld(const double *star_xy, const double *masses, int64_t N, double kappa_s,
                     double gamma, double phi_index, double num_phi_total,
                     const double *points, int64_t P, double *out)
{
    if (N < 1 || P < 0) return -2;
    residuals_ld(star_xy, masses, N, kappa_s, gamma, phi_index, num_phi_total, points, P, out);
    return 0;
}

int orc_residuals(const double *star_xy, const double *masses, int64_t N, double kappa_s,
                  double gamma, double phi_index, double num_phi_total,
                  const double *points, int64_t P, double *out)
{
    if (N < 1 || P < 0) return -2;
    residuals_d(star_xy, masses, N, kappa_s, gamma, phi_index, num_phi_total, points, P, out);
    return 0;
}

/* S1, S2, S3, Sm at given points (double / long double accumulation). */
int orc_star_sums(const double *star_xy, const double *masses, int64_t N, const double *points,
                  int64_t P, double *out)
{
    if (N < 1 || P < 0) return -2;
    star_sums_at_d(star_xy, masses, N, points, P, out);
    return 0;
}

int orc_star_sums_ld(const double *star_xy, const double *masses, int64_t N, const double *points,
                     int64_t P, double *out)
{
    if (N < 1 || P < 0) return -2;
    star_sums_at_ld(star_xy, masses, N, points, P, out);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Root-set matching (BASELINE.json north_star: "root sets per phase are compared after optimal
 * nearest-neighbour matching").  Brute force: for each a_i the nearest b_j over all j.  If
 * i -> j(i) is a bijection it is a perfect matching in which every a_i has its smallest
 * possible distance, so its maximum distance is the bottleneck-optimal one.
 *   out_max_err[s]   = max_i |a_i - b_j(i)|
 *   out_bijective[s] = 1 iff j(.) is a bijection and every pair has |a-b| <= rel_tol (1+|b|)
 * ---------------------------------------------------------------------------------------- */
int orc_match_root_sets(const double *a, const double *b, int64_t S, int64_t n, double rel_tol,
                        double *out_max_err, int32_t *out_bijective)
{
    if (S < 0 || n < 1) return -2;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t s = 0; s < S; ++s) {
        const double *as = a + 2 * s * n, *bs = b + 2 * s * n;
        int32_t *hits = (int32_t *)calloc((size_t)n, sizeof(int32_t));
        double max_err = 0.0;
        int ok = 1;
        for (int64_t i = 0; i < n; ++i) {
            double best = INFINITY;
            int64_t bj = -1;
            for (int64_t j = 0; j < n; ++j) {
                double dx = as[2 * i] - bs[2 * j], dy = as[2 * i + 1] - bs[2 * j + 1];
                double d2 = dx * dx + dy * dy;
                if (d2 < best) { best = d2; bj = j; }
            }
            if (bj < 0) { ok = 0; max_err = INFINITY; continue; } /* NaN input */
            double dist = sqrt(best);
            if (dist > max_err) max_err = dist;
            hits[bj] += 1;
            double bn = hypot(bs[2 * bj], bs[2 * bj + 1]);
            if (!(dist <= rel_tol * (1.0 + bn))) ok = 0;
        }
        for (int64_t j = 0; j < n; ++j) if (hits[j] != 1) ok = 0;
        free(hits);
        out_max_err[s] = max_err;
        out_bijective[s] = ok;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Completeness certificate of a claimed root set (SURVEY.md 8(c) pin P5; BASELINE.json north_star: "exactly
 * the paper's degree of distinct roots per phase").  P(z; phi) = F(z, phi) prod_i (z - z_i)^2 has
 * degree 2N with leading coefficient -c(phi), c = (1 - kappa_s) e^{-i phi} - gamma; expanding its two next
 * coefficients gives Vieta's sums of the 2N roots:
 *   sum_k z_k = 2 sum_i z_i,     sum_k z_k^2 = 2 sum_i z_i^2 + 2 (sum_i m_i) / c(phi).
 * A duplicated, missing or misplaced root breaks the first by its displacement.  Per row j,
 * phi_j = 2 pi (j + j_offset)/num_phi_total, straight long double sums:
 *   out_e1[j] = |sum z_k - 2 sum z_i| / sum |z_k|,
 *   out_e2[j] = |sum z_k^2 - 2 sum z_i^2 - 2 M / c_j| / sum |z_k|^2.
 * ---------------------------------------------------------------------------------------- */
int orc_vieta_residuals(const double *star_xy, const double *masses, int64_t N, double kappa_s, double gamma,
                        const double *roots, int64_t num_phi, int64_t j_offset, int64_t num_phi_total,
                        double *out_e1, double *out_e2)
{
    if (N < 1 || num_phi < 1 || num_phi_total < 1) return -2;
    long double complex sz = 0, sz2 = 0;
    long double M = 0;
    for (int64_t i = 0; i < N; ++i) {
        const long double complex zi = (long double)star_xy[2 * i] + I * (long double)star_xy[2 * i + 1];
        sz += zi;
        sz2 += zi * zi;
        M += masses[i];
    }
    const long double two_pi = 6.283185307179586476925286766559L;
    for (int64_t j = 0; j < num_phi; ++j) {
        const long double phi = two_pi * (long double)(j + j_offset) / (long double)num_phi_total;
        const long double complex c = (1.0L - (long double)kappa_s) * (cosl(phi) - I * sinl(phi)) - (long double)gamma;
        long double complex s1 = 0, s2 = 0;
        long double a1 = 0, a2 = 0;
        for (int64_t k = 0; k < 2 * N; ++k) {
            const long double complex z = (long double)roots[2 * (j * 2 * N + k)] + I * (long double)roots[2 * (j * 2 * N + k) + 1];
            s1 += z;
            s2 += z * z;
            a1 += cabsl(z);
            a2 += cabsl(z) * cabsl(z);
        }
        out_e1[j] = (double)(cabsl(s1 - 2.0L * sz) / a1);
        out_e2[j] = (double)(cabsl(s2 - 2.0L * sz2 - 2.0L * M / c) / a2);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Rectangular field of microlenses (Section 4.2, Appendix A at :386-401 and
 * Appendix B at :405-457).  The smooth term alpha_s(z) of a rectangular sheet with corner
 * c = c1 + i c2, its logarithms Taylor-expanded about the origin and truncated at power t
 * (Eq. B1-B2), the finite sheet extended to an infinite one.  Written as printed,
 * with the four corners c, conj c, -c, -conj c, their signs +,-,+,-, and principal logarithms:
 *   B2: alpha_s = -kappa_star i/pi [ sum_k sg_k (c_k - zb)(log c_k - sum_{j=1}^t (zb/c_k)^j / j) ]
 *                 - kappa_star (c + conj c + zb + z),                                 zb = conj z
 *   B7: d alpha_s/d zb = -kappa_star i/pi [ zb^t (1+(-1)^t)(1/c^t - 1/cb^t)
 *                 + sum_{j=1}^t zb^j (1+(-1)^j)(1/c^j - 1/cb^j)/j ] + kappa_star - 4 kappa_star atan(c2/c1)/pi
 *   B9: d2 alpha_s/d zb2 = -kappa_star i/(pi zb) [ t (zb/c)^t (1+(-1)^t)(1 - e^{2 i t Arg c})
 *                 + sum_{j=1}^t (zb/c)^j (1+(-1)^j)(1 - e^{2 i j Arg c}) ]
 *   B6: d alpha_s/d z = -kappa_star.
 * Then Eq. 15: F = gamma + S2 - conj(d alpha_s/d zb) - (1 - kappa - d alpha_s/d z) e^{-i phi},
 * F' = -2 S3 - conj(d2 alpha_s/d zb2), and Eq. 12: w = (1-kappa) z + gamma zb - conj(Sm) - alpha_s.
 * With t odd the polynomial has 2N + t - 1 roots.  double complex only.
 * ---------------------------------------------------------------------------------------- */
typedef double complex dcx;
#ifndef M_PI
#define M_PI 3.14159265358979323846264338327950288
#endif

static dcx rect_alpha_B2(double kappa_star, dcx c, int t, dcx z)
{
    const dcx zb = conj(z);
    const dcx corner[4] = {c, conj(c), -c, -conj(c)};
    const double sg[4] = {1.0, -1.0, 1.0, -1.0};
    dcx sum = 0;
    for (int k = 0; k < 4; ++k) {
        dcx series = 0, q = 1;
        for (int j = 1; j <= t; ++j) {
            q *= zb / corner[k];
            series += q / (double)j;
        }
        sum += sg[k] * (corner[k] - zb) * (clog(corner[k]) - series);
    }
    return -kappa_star * I / M_PI * sum - kappa_star * (c + conj(c) + zb + z);
}

static dcx rect_dalpha_dzbar_B7(double kappa_star, dcx c, int t, dcx z)
{
    const dcx zb = conj(z), cb = conj(c);
    const double sign_t = (t % 2 == 0) ? 2.0 : 0.0;   /* 1 + (-1)^t */
    dcx sum = cpow(zb, t) * sign_t * (1.0 / cpow(c, t) - 1.0 / cpow(cb, t));
    dcx zp = 1, cp = 1, cbp = 1;
    for (int j = 1; j <= t; ++j) {
        zp *= zb; cp *= c; cbp *= cb;
        const double sign_j = (j % 2 == 0) ? 2.0 : 0.0;
        sum += zp * sign_j * (1.0 / cp - 1.0 / cbp) / (double)j;
    }
    return -kappa_star * I / M_PI * sum + kappa_star - 4.0 * kappa_star * atan(cimag(c) / creal(c)) / M_PI;
}

static dcx rect_d2alpha_dzbar2_B9(double kappa_star, dcx c, int t, dcx z)
{
    const dcx zb = conj(z);
    const double argc = carg(c);
    const double sign_t = (t % 2 == 0) ? 2.0 : 0.0;
    dcx sum = (double)t * cpow(zb / c, t) * sign_t * (1.0 - cexp(I * 2.0 * argc * (double)t));
    dcx q = 1;
    for (int j = 1; j <= t; ++j) {
        q *= zb / c;
        const double sign_j = (j % 2 == 0) ? 2.0 : 0.0;
        sum += q * sign_j * (1.0 - cexp(I * 2.0 * argc * (double)j));
    }
    return -kappa_star * I / (M_PI * zb) * sum;
}

int orc_rect_sheet(double kappa_star, double c1, double c2, int t, const double *points, int64_t P,
                   double *out_alpha, double *out_dzbar, double *out_d2zbar)
{
    if (!(c1 > 0) || !(c2 > 0) || t < 1 || P < 0) return -2;
    const dcx c = c1 + I * c2;
    for (int64_t p = 0; p < P; ++p) {
        const dcx z = points[2 * p] + I * points[2 * p + 1];
        const dcx a = rect_alpha_B2(kappa_star, c, t, z), b = rect_dalpha_dzbar_B7(kappa_star, c, t, z),
                  d = rect_d2alpha_dzbar2_B9(kappa_star, c, t, z);
        if (out_alpha) { out_alpha[2 * p] = creal(a); out_alpha[2 * p + 1] = cimag(a); }
        if (out_dzbar) { out_dzbar[2 * p] = creal(b); out_dzbar[2 * p + 1] = cimag(b); }
        if (out_d2zbar) { out_d2zbar[2 * p] = creal(d); out_d2zbar[2 * p + 1] = cimag(d); }
    }
    return 0;
}

/* Truncation power t for a wanted error eps of alpha_s inside |z| <= |c|/s (Eq. B5):
 * the smallest odd t with kappa_star/pi * 4/(t+1) * s^-(t+1) * |c| (s+1)/(s-1) <= eps, then raised by 2
 * until (t-1) Arg c mod pi is at least 10 % of pi away from 0 and pi.                  */
int orc_rect_truncation(double kappa_star, double c1, double c2, double s, double eps)
{
    if (!(s > 1.0) || !(eps > 0.0)) return -2;
    const double cabs_ = hypot(c1, c2), argc = atan2(c2, c1);
    int t = 1;
    while (kappa_star / M_PI * 4.0 / (t + 1) * pow(1.0 / s, t + 1) * cabs_ * (s + 1) / (s - 1) > eps && t < 2001) t += 2;
    for (int guard = 0; guard < 1000; ++guard) {
        double r = fmod((t - 1) * argc, M_PI);
        if (r >= 0.1 * M_PI && r <= 0.9 * M_PI) break;
        t += 2;
    }
    return t;
}

/* One Aberth-Ehrlich solve for one phase with the rectangular sheet: aberth_row of
 * aberth_generic.inc with F and F' extended as above; n_r = 2N + t - 1.                           */
static int aberth_row_rect(const double *star_xy, const double *masses, int64_t N, double kappa_s,
                           double gamma, double kappa_star, dcx c, int t, double phi, double tol,
                           int max_iter, int64_t n_r, dcx *z, dcx *znew, unsigned char *frozen,
                           int64_t *n_unconverged)
{
    const dcx rot = (1 - kappa_s) * (cos(phi) - I * sin(phi));   /* (1 - kappa - d alpha_s/dz) e^{-i phi}, B6 */
    memset(frozen, 0, (size_t)n_r);
    int iters = 0;
    int64_t n_active = n_r;
    while (n_active > 0 && iters < max_iter) {
#pragma omp parallel for schedule(dynamic, 16)
        for (int64_t k = 0; k < n_r; ++k) {
            if (frozen[k]) { znew[k] = z[k]; continue; }
            dcx S1, S2, S3, Sm;
            star_sums_d(star_xy, masses, N, z[k], &S1, &S2, &S3, &Sm);
            dcx A = 0;
            for (int64_t r = 0; r < n_r; ++r) {
                if (r == k) continue;
                A += cinv_d(z[k] - z[r]);
            }
            dcx F = gamma + S2 - conj(rect_dalpha_dzbar_B7(kappa_star, c, t, z[k])) - rot;
            dcx Fp = -2 * S3 - conj(rect_d2alpha_dzbar2_B9(kappa_star, c, t, z[k]));
            /* P'/P = F'/F + 2 S1 (Eq. 19): the extra t - 1 roots come from the polynomial part of F alone */
            dcx Delta = F / (Fp + F * (2 * S1 - A));
            znew[k] = z[k] - Delta;
            if (cabs(Delta) < tol) frozen[k] = 2;
        }
        n_active = 0;
        for (int64_t k = 0; k < n_r; ++k) {
            z[k] = znew[k];
            if (frozen[k] == 2) frozen[k] = 1;
            if (!frozen[k]) ++n_active;
        }
        ++iters;
    }
    *n_unconverged = n_active;
    return iters;
}

/* Rows of the phase grid for the rectangular sheet.  Cold start: z_i +/- 1 "plus an additional number
 * as required from alpha_s(z) evenly spread in a circle around the microlenses": the
 * t - 1 extra seeds at seed_radius e^{2 pi i (k + 1/2)/(t-1)} (radius: DESIGN.md reading R25).       */
int orc_rect_critical_curve_rows(const double *star_xy, const double *masses, int64_t N, double kappa_s,
                                 double gamma, double kappa_star, double c1, double c2, int t,
                                 double seed_radius, int64_t num_phi_total, const int64_t *rows,
                                 int64_t nrows, double tol, int max_iter, const double *init_roots,
                                 double *out_roots, int32_t *out_iters, int32_t *out_unconverged)
{
    if (N < 1 || num_phi_total < 1 || nrows < 0 || t < 1 || (t % 2) == 0) return -2;
    const int64_t n_r = 2 * N + t - 1;
    const dcx c = c1 + I * c2;
    dcx *z = (dcx *)malloc(sizeof(dcx) * (size_t)n_r), *znew = (dcx *)malloc(sizeof(dcx) * (size_t)n_r);
    unsigned char *frozen = (unsigned char *)malloc((size_t)n_r);
    if (!z || !znew || !frozen) { free(z); free(znew); free(frozen); return -1; }
    if (init_roots) {
        for (int64_t k = 0; k < n_r; ++k) z[k] = init_roots[2 * k] + I * init_roots[2 * k + 1];
    } else {
        cold_seeds_d(star_xy, N, z);
        for (int64_t k = 0; k < t - 1; ++k) {
            const double ang = 2.0 * M_PI * ((double)k + 0.5) / (double)(t - 1);
            z[2 * N + k] = seed_radius * (cos(ang) + I * sin(ang));
        }
    }
    for (int64_t q = 0; q < nrows; ++q) {
        const double phi = 2.0 * M_PI * (double)rows[q] / (double)num_phi_total;
        int64_t unconv = 0;
        int it = aberth_row_rect(star_xy, masses, N, kappa_s, gamma, kappa_star, c, t, phi, tol, max_iter, n_r,
                                 z, znew, frozen, &unconv);
        for (int64_t k = 0; k < n_r; ++k) {
            out_roots[2 * (q * n_r + k)] = creal(z[k]);
            out_roots[2 * (q * n_r + k) + 1] = cimag(z[k]);
        }
        if (out_iters) out_iters[q] = it;
        if (out_unconverged) out_unconverged[q] = (int32_t)unconv;
    }
    free(z); free(znew); free(frozen);
    return 0;
}

/* Caustic points with the rectangular sheet: Eq. 12 with alpha_s of Eq. B2 and
 * kappa = kappa_s + kappa_star:  w = (1-kappa) z + gamma conj z - sum m_i/(conj z - conj z_i) - alpha_s(z). */
int orc_rect_caustics(const double *star_xy, const double *masses, int64_t N, double kappa_s, double gamma,
                      double kappa_star, double c1, double c2, int t, const double *points, int64_t P,
                      double *out)
{
    if (N < 1 || P < 0 || t < 1) return -2;
    const dcx c = c1 + I * c2;
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < P; ++p) {
        const dcx z = points[2 * p] + I * points[2 * p + 1];
        dcx defl = 0;
        for (int64_t i = 0; i < N; ++i) {
            const dcx zi = star_xy[2 * i] + I * star_xy[2 * i + 1];
            defl += masses[i] * cinv_d(conj(z) - conj(zi));
        }
        const dcx w = (1 - (kappa_s + kappa_star)) * z + gamma * conj(z) - defl - rect_alpha_B2(kappa_star, c, t, z);
        out[2 * p] = creal(w);
        out[2 * p + 1] = cimag(w);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Chain joining (fn. 5 at :217): "the start of one chain is the end of another, with
 * chains joining together until closed loops are formed".  Row s of `rows` holds the n roots of
 * phase s in any column order; out_next[s][i] is the column of row (s+1) mod S whose root is nearest
 * to root i of row s (brute force over all columns; the first index wins a tie).  Roots move
 * continuously with phi, so for a fine enough grid that root continues the chain.
 *   out_bijective[s] = 1 iff i -> out_next[s][i] is a bijection (every chain has one successor).
 * ---------------------------------------------------------------------------------------- */
int orc_link_rows(const double *rows, int64_t S, int64_t n, int32_t *out_next, int32_t *out_bijective)
{
    if (S < 1 || n < 1) return -2;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t s = 0; s < S; ++s) {
        const double *as = rows + 2 * s * n, *bs = rows + 2 * ((s + 1) % S) * n;
        int32_t *hits = (int32_t *)calloc((size_t)n, sizeof(int32_t));
        int ok = 1;
        for (int64_t i = 0; i < n; ++i) {
            double best = INFINITY;
            int64_t bj = -1;
            for (int64_t j = 0; j < n; ++j) {
                double dx = as[2 * i] - bs[2 * j], dy = as[2 * i + 1] - bs[2 * j + 1];
                double d2 = dx * dx + dy * dy;
                if (d2 < best) { best = d2; bj = j; }
            }
            out_next[s * n + i] = (int32_t)bj;
            if (bj < 0) ok = 0; else hits[bj] += 1;
        }
        for (int64_t j = 0; j < n; ++j) if (hits[j] != 1) ok = 0;
        out_bijective[s] = ok;
        free(hits);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Number of caustic crossings per source pixel (Section 5.1): "Since the caustics
 * are oriented curves, winding numbers provide the number of caustic crossings.  For every
 * (pixelized) source location, we use ... Sunday's (2001) algorithm to calculate the winding number
 * of the discretized caustic polygons around that point".  The polygons are the chains of caustic
 * points joined by `next` (NULL = column i continues in column i), closed from row S-1 back to
 * row 0.  The caustics are traced clockwise, so the count is MINUS the usual
 * counter-clockwise winding number (reading R21).
 * Written as the definition: for each pixel centre, a loop over every segment with Sunday's
 * crossing rule (an upward edge with the point strictly on its left adds one, a downward edge
 * with the point strictly on its right subtracts one).  Pixel (ix, iy) has its centre at
 * (x0 + (ix + 1/2) pixel, y0 + (iy + 1/2) pixel); out_map is [ny][nx] row-major.
 * out_ambiguous (may be NULL), [ny][nx]: 1 where the centre lies within 1e-9 pixel of a segment it
 * could cross, so that rounding may decide the count there.
 * ---------------------------------------------------------------------------------------- */
int orc_crossing_map(const double *caustics, const int32_t *next, int64_t S, int64_t n,
                     double x0, double y0, double pixel, int32_t nx, int32_t ny,
                     int32_t *out_map, uint8_t *out_ambiguous)
{
    if (S < 1 || n < 1 || nx < 1 || ny < 1 || !(pixel > 0.0)) return -2;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t pix = 0; pix < (int64_t)nx * ny; ++pix) {
        const int64_t iy = pix / nx, ix = pix % nx;
        const long double px = (long double)x0 + ((long double)ix + 0.5L) * (long double)pixel;
        const long double py = (long double)y0 + ((long double)iy + 0.5L) * (long double)pixel;
        int32_t wn = 0;
        int amb = 0;
        for (int64_t s = 0; s < S; ++s) {
            const double *a = caustics + 2 * s * n, *b = caustics + 2 * ((s + 1) % S) * n;
            for (int64_t i = 0; i < n; ++i) {
                const int64_t j = next ? next[s * n + i] : i;
                if (j < 0) continue;
                const long double ax = a[2 * i], ay = a[2 * i + 1], bx = b[2 * j], by = b[2 * j + 1];
                if (!(ax == ax && ay == ay && bx == bx && by == by)) continue;   /* NaN point: no segment */
                /* isLeft > 0: (px,py) left of the directed line a -> b */
                const long double is_left = (bx - ax) * (py - ay) - (px - ax) * (by - ay);
                if (ay <= py) {
                    if (by > py && is_left > 0) ++wn;          /* upward crossing, point on the left  */
                } else {
                    if (by <= py && is_left < 0) --wn;         /* downward crossing, point on the right */
                }
                if (out_ambiguous) {
                    const long double lo = ay < by ? ay : by, hi = ay < by ? by : ay;
                    const long double len = sqrtl((bx - ax) * (bx - ax) + (by - ay) * (by - ay));
                    const long double eps = 1e-9L * (long double)pixel;
                    if (py >= lo - eps && py <= hi + eps && fabsl(is_left) <= eps * (len + eps)) amb = 1;
                    if (fabsl(py - ay) <= eps || fabsl(py - by) <= eps) {
                        /* the ray grazes an end point: which of the two segments there counts is a
                           rounding decision if the point is also to the left of it */
                        amb = amb || (px <= (ax > bx ? ax : bx) + eps);
                    }
                }
            }
        }
        out_map[pix] = -wn;
        if (out_ambiguous) out_ambiguous[pix] = (uint8_t)amb;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Chains and closed loops ("Every one of the initial n_r roots begins and ends a
 * 'chain' of values from 0 to 2 pi ... sometimes 2 or more chains are needed to fully create a closed
 * critical curve"; fn. 5 at :217: "the start of one chain is the end of another, with chains joining
 * together until closed loops are formed").  `next` is the successor table of orc_link_rows.
 * Chain k is the one that starts in column k of row 0; written as the definition:
 *   chain_col[0][k] = k,  chain_col[s+1][k] = next[s][chain_col[s][k]],
 *   chain_end[k]    = next[S-1][chain_col[S-1][k]]   (the column of row 0 the chain arrives at after
 *                     the whole turn of phi: the start of the chain that continues it),
 *   loop_id[k]      = the smallest chain index met by walking k -> chain_end[k] -> ... back to k,
 *   num_loops       = number of distinct loop_id values.
 * A chain that meets an entry outside [0, n) gets -1 from there on, chain_end = -1 and loop_id = -1;
 * so does a chain whose walk does not return to it within n steps (chain_end not a bijection).
 * out_chain_col may be NULL.
 * ---------------------------------------------------------------------------------------- */
int orc_closed_loops(const int32_t *next, int64_t S, int64_t n, int32_t *out_chain_col,
                     int32_t *out_chain_end, int32_t *out_loop_id, int32_t *out_num_loops)
{
    if (S < 1 || n < 1) return -2;
    for (int64_t k = 0; k < n; ++k) {
        int64_t c = k;
        for (int64_t s = 0; s < S; ++s) {
            if (out_chain_col) out_chain_col[s * n + k] = (int32_t)c;
            if (c >= 0) {
                c = next[s * n + c];
                if (c < 0 || c >= n) c = -1;
            }
        }
        out_chain_end[k] = (int32_t)c;
    }
    int32_t loops = 0;
    for (int64_t k = 0; k < n; ++k) {
        int64_t c = k, smallest = k, steps = 0;
        int closed = 0;
        while (steps < n) {
            c = out_chain_end[c];
            ++steps;
            if (c < 0) break;
            if (c == k) { closed = 1; break; }
            if (c < smallest) smallest = c;
        }
        out_loop_id[k] = closed ? (int32_t)smallest : -1;
        if (closed && smallest == k) ++loops;
    }
    *out_num_loops = loops;
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Distance to the nearest caustic for an expanding source (Section 5.2, Fig. 5 top):
 * "the distance from each pixel to the nearest caustic ... calculated from the map of N_caustic
 * crossings using a Euclidean distance transform".  Reading (R28): a pixel is a caustic
 * pixel if one of its 4 neighbours inside the map holds a different count; the distance of pixel p is
 * pixel * min over caustic pixels q of |p - q| (centre to centre, 0 on a caustic pixel), +inf if the map
 * has no caustic pixel.  Brute force over all pairs, squared distances in integers.
 * out_d2 (may be NULL): the squared distance in pixels as int64 (-1 for +inf).
 * ---------------------------------------------------------------------------------------- */
static int caustic_pixel(const int32_t *map, int64_t nx, int64_t ny, int64_t x, int64_t y)
{
    const int32_t v = map[y * nx + x];
    if (x > 0 && map[y * nx + x - 1] != v) return 1;
    if (x + 1 < nx && map[y * nx + x + 1] != v) return 1;
    if (y > 0 && map[(y - 1) * nx + x] != v) return 1;
    if (y + 1 < ny && map[(y + 1) * nx + x] != v) return 1;
    return 0;
}

int orc_distance_map(const int32_t *map, int32_t nx, int32_t ny, double pixel, double *out, int64_t *out_d2)
{
    if (nx < 1 || ny < 1 || !(pixel > 0.0)) return -2;
    const int64_t P = (int64_t)nx * ny;
    uint8_t *edge = (uint8_t *)malloc((size_t)P);
    for (int64_t y = 0; y < ny; ++y)
        for (int64_t x = 0; x < nx; ++x) edge[y * nx + x] = (uint8_t)caustic_pixel(map, nx, ny, x, y);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t p = 0; p < P; ++p) {
        const int64_t py = p / nx, px = p % nx;
        int64_t best = -1;
        for (int64_t qy = 0; qy < ny; ++qy)
            for (int64_t qx = 0; qx < nx; ++qx) {
                if (!edge[qy * nx + qx]) continue;
                const int64_t d2 = (px - qx) * (px - qx) + (py - qy) * (py - qy);
                if (best < 0 || d2 < best) best = d2;
            }
        if (out_d2) out_d2[p] = best;
        out[p] = best < 0 ? INFINITY : pixel * sqrt((double)best);
    }
    free(edge);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Distance to the nearest caustic for a source moving along a direction (Fig. 5
 * bottom, Fig. 6-7).  Reading (R29): the direction is the integer vector u = (ux, uy); the ray
 * starts at the centre of pixel p; the caustic is met where the ray first enters (the open interior
 * of) a pixel whose count differs from that of p; the distance is from the centre of p to that entry
 * point.  If the ray leaves the map first, the value is MINUS the distance to the exit point: a lower
 * bound only ("the border of the map is a boundary that can be hit in the distance algorithms despite
 * not being a caustic", Fig. 5 caption at PAPER.md:245).
 * Written as the definition: for each pixel p a loop over every other pixel q with a different count,
 * ray/square intersection by the slab rule in exact rational arithmetic (coordinates doubled so that
 * centres are even and pixel borders odd integers), the smallest entry parameter wins.
 * ---------------------------------------------------------------------------------------- */
typedef struct { int64_t num, den; } orc_rat;            /* den > 0;  +-inf as (+-1, 0) */
static int rat_lt(orc_rat a, orc_rat b)                   /* a < b */
{
    if (a.den == 0 && b.den == 0) return a.num < b.num;
    if (a.den == 0) return a.num < 0;
    if (b.den == 0) return b.num > 0;
    return a.num * b.den < b.num * a.den;
}
static orc_rat rat_make(int64_t num, int64_t den)
{
    orc_rat r;
    if (den < 0) { num = -num; den = -den; }
    r.num = num; r.den = den;
    return r;
}
/* parameter interval (lo, hi) of o + t u inside the open slab (a, b) along one axis; returns 0 if empty */
static int slab(int64_t o, int64_t u, int64_t a, int64_t b, orc_rat *lo, orc_rat *hi)
{
    if (u == 0) {
        if (!(a < o && o < b)) return 0;
        *lo = rat_make(-1, 0); *hi = rat_make(1, 0);
        return 1;
    }
    orc_rat ta = rat_make(a - o, u), tb = rat_make(b - o, u);
    if (rat_lt(tb, ta)) { orc_rat t = ta; ta = tb; tb = t; }
    *lo = ta; *hi = tb;
    return 1;
}

int orc_directional_distance_map(const int32_t *map, int32_t nx, int32_t ny, double pixel, int32_t ux, int32_t uy,
                                 double *out)
{
    if (nx < 1 || ny < 1 || !(pixel > 0.0) || (ux == 0 && uy == 0)) return -2;
    const int64_t P = (int64_t)nx * ny;
    const double ulen = sqrt((double)((int64_t)ux * ux + (int64_t)uy * uy));
    const orc_rat zero = rat_make(0, 1);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t p = 0; p < P; ++p) {
        const int64_t py = p / nx, px = p % nx;
        const int64_t ox = 2 * px, oy = 2 * py;
        const int32_t v = map[p];
        int found = 0;
        orc_rat best = rat_make(1, 0);
        for (int64_t qy = 0; qy < ny; ++qy)
            for (int64_t qx = 0; qx < nx; ++qx) {
                if (map[qy * nx + qx] == v) continue;
                orc_rat xl, xh, yl, yh;
                if (!slab(ox, ux, 2 * qx - 1, 2 * qx + 1, &xl, &xh)) continue;
                if (!slab(oy, uy, 2 * qy - 1, 2 * qy + 1, &yl, &yh)) continue;
                const orc_rat enter = rat_lt(xl, yl) ? yl : xl;      /* max of the lows  */
                const orc_rat leave = rat_lt(xh, yh) ? xh : yh;      /* min of the highs */
                if (!rat_lt(enter, leave)) continue;                   /* touches a corner or misses */
                if (!rat_lt(zero, leave)) continue;                    /* behind the start */
                if (!rat_lt(zero, enter)) continue;                    /* q == p cannot happen (same count) */
                if (!found || rat_lt(enter, best)) { best = enter; found = 1; }
            }
        if (found) {
            out[p] = pixel * 0.5 * ulen * ((double)best.num / (double)best.den);
        } else {
            /* exit point of the map rectangle (-1, 2 nx - 1) x (-1, 2 ny - 1) */
            orc_rat xl, xh, yl, yh;
            slab(ox, ux, -1, 2 * (int64_t)nx - 1, &xl, &xh);
            slab(oy, uy, -1, 2 * (int64_t)ny - 1, &yl, &yh);
            const orc_rat leave = rat_lt(xh, yh) ? xh : yh;
            out[p] = -(pixel * 0.5 * ulen * ((double)leave.num / (double)leave.den));
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Distribution of the distance to the nearest caustic (Fig. 6: "probability distribution of
 * the distance to the nearest caustic" per direction of motion; Fig. 7: the same split by "where the source
 * happens to lie in the map of N_caustic crossings").  A histogram of a distance map: pixel p with a finite
 * distance d >= 0 (a negative value of the moving-source map is limited by the border of the map and is left
 * out, so is +inf) is counted in bin floor(d / bin_width) if that is < num_bins, in row
 * min(max(count_p, 0), num_counts - 1) of the table (row 0 if there is no crossing map).
 * out_hist [num_counts][num_bins] int64; out_left_out [1] int64 = pixels not counted.
 * ---------------------------------------------------------------------------------------- */
int orc_distance_histogram(const double *distance, const int32_t *crossing_map, int64_t num_pixels, double bin_width,
                           int32_t num_bins, int32_t num_counts, int64_t *out_hist, int64_t *out_left_out)
{
    if (num_pixels < 0 || !(bin_width > 0.0) || num_bins < 1 || num_counts < 1) return -2;
    for (int64_t i = 0; i < (int64_t)num_bins * num_counts; ++i) out_hist[i] = 0;
    int64_t left = 0;
    for (int64_t p = 0; p < num_pixels; ++p) {
        const double d = distance[p];
        if (!(d >= 0.0) || d == INFINITY) { ++left; continue; }
        const double b = floor(d / bin_width);
        if (!(b < (double)num_bins)) { ++left; continue; }
        int32_t row = crossing_map ? crossing_map[p] : 0;
        if (row < 0) row = 0;
        if (row > num_counts - 1) row = num_counts - 1;
        out_hist[(int64_t)row * num_bins + (int64_t)b] += 1;
    }
    if (out_left_out) *out_left_out = left;
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Star-field generator (recipe in DESIGN.md "Input recipe").
 * Counter-based Philox4x32-10 (Salmon, Moraes, Dror & Shaw 2011, "Parallel random numbers:
 * as easy as 1, 2, 3"), restated from the published algorithm.
 * ---------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* two 32-bit words -> uniform in [0,1) with 53 bits */
static double u53(uint32_t hi, uint32_t lo)
{
    uint64_t bits = ((uint64_t)hi << 32) | (uint64_t)lo;
    return (double)(bits >> 11) * (1.0 / 9007199254740992.0);
}

/* Inverse CDF of dN/dm ∝ m^-alpha on [lo, hi]. */
static double powerlaw_icdf(double u, double lo, double hi, double alpha)
{
    if (alpha == 1.0) return lo * pow(hi / lo, u);
    double e = 1.0 - alpha;
    double a = pow(lo, e), b = pow(hi, e);
    return pow(a + u * (b - a), 1.0 / e);
}

/* mass_model: 0 equal masses (m = 1)
 *             1 single power law, params = {m_lo, m_hi, alpha}         (default 0.08, 1, 2.35)
 *             2 three-segment broken power law, continuous at the breaks,
 *               params = {m0, m1, m2, m3, alpha1, alpha2, alpha3}       (default 0.01, 0.08, 0.5, 1.5,
 *                                                                        0.3, 1.3, 2.3)
 * Masses are divided by the sample mean, so sum m_i = N and theta_star is the Einstein radius of
 * the mean mass (BASELINE.json configs[2]).  Positions are uniform in the disk of radius
 * R = sqrt(sum m_i / kappa_star) = sqrt(N / kappa_star)  (Eq. 9, with A_star = pi R^2),
 * by rejection from the square: star i, attempt a uses Philox counter (i_lo, i_hi, a, 0) and key
 * (seed_lo, seed_hi); x = 2 u53(r0, r1) - 1, y = 2 u53(r2, r3) - 1, accepted iff x*x + y*y < 1.
 * The mass of star i uses counter (i_lo, i_hi, 0, 1) and u = u53(r0, r1).                       */
static int star_field_any(uint64_t seed, int64_t N, double kappa_star, int mass_model, const double *mass_params,
                          double aspect, double *star_xy, double *masses, double *out_radius, double *out_corner);

int orc_star_field(uint64_t seed, int64_t N, double kappa_star, int mass_model,
                   const double *mass_params, double *star_xy, double *masses, double *out_radius)
{
    return star_field_any(seed, N, kappa_star, mass_model, mass_params, 0.0, star_xy, masses, out_radius, NULL);
}

/* Rectangular field (Section 4.2; Appendix A at :386: stars in the rectangle with corner
 * c = c1 + i c2).  Same masses; Eq. 9 with A_star = 4 c1 c2 and sum m_i = N gives
 * c2 = sqrt(pi N / (4 kappa_star aspect)), c1 = aspect c2.  Star i sits at (c1 x, c2 y) with the x, y of
 * attempt 0 of the disk recipe (uniform in [-1,1)^2, no rejection).  out_corner = {c1, c2}.              */
int orc_star_field_rect(uint64_t seed, int64_t N, double kappa_star, double aspect, int mass_model,
                        const double *mass_params, double *star_xy, double *masses, double *out_corner)
{
    if (!(aspect > 0.0) || !(aspect < INFINITY)) return -2;
    return star_field_any(seed, N, kappa_star, mass_model, mass_params, aspect, star_xy, masses, NULL, out_corner);
}

static int star_field_any(uint64_t seed, int64_t N, double kappa_star, int mass_model, const double *mass_params,
                          double aspect, double *star_xy, double *masses, double *out_radius, double *out_corner)
{
    if (N < 1 || !(kappa_star > 0.0) || mass_model < 0 || mass_model > 2) return -2;
    static const double salpeter[3] = {0.08, 1.0, 2.35};
    static const double kroupa[7] = {0.01, 0.08, 0.5, 1.5, 0.3, 1.3, 2.3};
    const double *p = mass_params;
    if (!p) p = (mass_model == 1) ? salpeter : kroupa;
    const uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};

    /* masses */
    double seg_prob[3] = {0, 0, 0}, seg_cum[4] = {0, 0, 0, 0};
    if (mass_model == 2) {
        /* segment s: dN/dm = A_s m^-alpha_s on [p[s], p[s+1]], A_1 = 1, continuity at the breaks */
        double A[3];
        A[0] = 1.0;
        A[1] = A[0] * pow(p[1], p[5] - p[4]);
        A[2] = A[1] * pow(p[2], p[6] - p[5]);
        double total = 0.0;
        for (int s = 0; s < 3; ++s) {
            double al = p[4 + s], lo = p[s], hi = p[s + 1];
            double integral = (al == 1.0) ? log(hi / lo) : (pow(hi, 1.0 - al) - pow(lo, 1.0 - al)) / (1.0 - al);
            seg_prob[s] = A[s] * integral;
            total += seg_prob[s];
        }
        for (int s = 0; s < 3; ++s) { seg_prob[s] /= total; seg_cum[s + 1] = seg_cum[s] + seg_prob[s]; }
        seg_cum[3] = 1.0;
    }
    double sum = 0.0;
    for (int64_t i = 0; i < N; ++i) {
        double m = 1.0;
        if (mass_model != 0) {
            uint32_t ctr[4] = {(uint32_t)((uint64_t)i & 0xFFFFFFFFu), (uint32_t)((uint64_t)i >> 32), 0u, 1u};
            uint32_t r[4];
            orc_philox4x32_10(ctr, key, r);
            double u = u53(r[0], r[1]);
            if (mass_model == 1) {
                m = powerlaw_icdf(u, p[0], p[1], p[2]);
            } else {
                int s = (u < seg_cum[1]) ? 0 : (u < seg_cum[2]) ? 1 : 2;
                double v = (u - seg_cum[s]) / seg_prob[s];
                m = powerlaw_icdf(v, p[s], p[s + 1], p[4 + s]);
            }
        }
        masses[i] = m;
        sum += m;
    }
    const double mean = sum / (double)N;
    for (int64_t i = 0; i < N; ++i) masses[i] /= mean;

    /* positions */
    if (aspect > 0.0) {
        const double c2 = sqrt(3.14159265358979323846 * (double)N / (4.0 * kappa_star * aspect));
        const double c1 = aspect * c2;
        for (int64_t i = 0; i < N; ++i) {
            uint32_t ctr[4] = {(uint32_t)((uint64_t)i & 0xFFFFFFFFu), (uint32_t)((uint64_t)i >> 32), 0u, 0u};
            uint32_t r[4];
            orc_philox4x32_10(ctr, key, r);
            star_xy[2 * i] = c1 * (2.0 * u53(r[0], r[1]) - 1.0);
            star_xy[2 * i + 1] = c2 * (2.0 * u53(r[2], r[3]) - 1.0);
        }
        if (out_corner) { out_corner[0] = c1; out_corner[1] = c2; }
        return 0;
    }
    const double R = sqrt((double)N / kappa_star);
    for (int64_t i = 0; i < N; ++i) {
        double x = 0.0, y = 0.0;
        int ok = 0;
        for (uint32_t attempt = 0; attempt < 256u && !ok; ++attempt) {
            uint32_t ctr[4] = {(uint32_t)((uint64_t)i & 0xFFFFFFFFu), (uint32_t)((uint64_t)i >> 32), attempt, 0u};
            uint32_t r[4];
            orc_philox4x32_10(ctr, key, r);
            x = 2.0 * u53(r[0], r[1]) - 1.0;
            y = 2.0 * u53(r[2], r[3]) - 1.0;
            ok = (x * x + y * y < 1.0);
        }
        if (!ok) return -3;
        star_xy[2 * i] = R * x;
        star_xy[2 * i + 1] = R * y;
    }
    if (out_radius) *out_radius = R;
    return 0;
}

int orc_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    n = omp_get_max_threads();
#endif
    return n;
}
