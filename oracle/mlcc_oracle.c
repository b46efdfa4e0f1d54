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
 * Philox known-answer vectors, generator statistics.
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
int orc_star_field(uint64_t seed, int64_t N, double kappa_star, int mass_model,
                   const double *mass_params, double *star_xy, double *masses, double *out_radius)
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
