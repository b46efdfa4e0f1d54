/* mlcc.h — C-ABI of the B200-native critical-curve / caustic library (libmlcc.so).
 *
 * Hot path of arXiv 2506.02121 ("A GPU Code for Finding Microlensing Critical Curves and
 * Caustics"), cited below as PAPER.md:<line>.  Lengths are in Einstein radii of the unit mass
 * (theta_star = 1).  The lens equation is Eq. 12 with the infinite
 * compensating sheet alpha_s(z) = -kappa_star z of Appendix A:
 *
 *     w = (1 - kappa_s) z + gamma conj(z) - sum_i m_i / (conj(z) - conj(z_i)),
 *     kappa_s = kappa - kappa_star   (smooth convergence),
 *
 * and the critical curves are the roots z of Eq. 15 for each phase phi:
 *
 *     F(z, phi) = gamma + sum_i m_i / (z - z_i)^2 - (1 - kappa_s) e^{-i phi} = 0,
 *
 * i.e. the 2N roots of P(z) = F(z) prod_i (z - z_i)^2 (Eq. 16).
 *
 * Conventions for every entry point
 *  - Complex numbers are interleaved (re, im) doubles; arrays of them must be 16-byte aligned.
 *  - Unless the name ends in _host, array pointers are DEVICE pointers to caller-owned,
 *    caller-allocated buffers (e.g. PyTorch tensors).  The library never frees or keeps them.
 *    Pointers documented "host" are host pointers.  _host entry points take HOST pointers for
 *    everything and do their own device allocation and host<->device copies.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Work is
 *    enqueued on it; calls that return a status computed on the device (convergence counts)
 *    synchronise that stream before returning.  Entry points without a stream argument use the
 *    default stream and synchronise it.
 *  - Workspace is allocated per call with the stream-ordered allocator and released before return.
 *    Side effect, process-wide: the first call on a device sets the release threshold of that device's
 *    DEFAULT CUDA memory pool to "keep" (cudaMemPoolAttrReleaseThreshold), so that the GB-sized scratch is
 *    not returned to the driver at every synchronisation.  Other cudaMallocAsync users of the same pool see
 *    their freed blocks cached as well; cudaMemPoolTrimTo releases them.
 *  - Return value: mlcc_status.  Errors never throw or exit; mlcc_last_error() gives the text
 *    of the last failure on the calling thread.
 *  - Thread-safety: re-entrant; concurrent calls must use distinct streams.
 */
#ifndef MLCC_H_
#define MLCC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum mlcc_status {
    MLCC_OK = 0,
    MLCC_ERR_INVALID_ARG = 1,   /* null pointer, N < 1, num_phi < 1, tol <= 0, max_iter < 1, non-finite
                                   kappa_s / gamma, or c(phi_j) = (1-kappa_s) e^{-i phi_j} - gamma = 0 on
                                   a grid row (the degree of P drops there)            */
    MLCC_ERR_CUDA = 2,          /* a CUDA call failed; text in mlcc_last_error()                       */
    MLCC_ERR_NOMEM = 3,         /* workspace allocation failed                                         */
    MLCC_ERR_NOT_CONVERGED = 4, /* some root hit max_iter; outputs are fully written, the counts are in
                                   out_unconverged                                                     */
    MLCC_ERR_DEGENERATE = 5     /* a NaN/Inf step: a root landed on a star or on another root, or two
                                   stars coincide; the offending roots are frozen where they were       */
} mlcc_status;

/* Mass models of the star-field generator (BASELINE.json configs; the paper names none). */
enum { MLCC_MASS_EQUAL = 0, MLCC_MASS_POWER_LAW = 1, MLCC_MASS_BROKEN_POWER_LAW = 2 };

/* How the star sums S1, S2, S3, Sm are evaluated (mlcc_options.star_sum_mode, mlcc_star_sums).
 * DIRECT: the O(N) sums over all stars as Eq. 15 / Eq. 19 are written (BASELINE.json north_star).
 * FMM:    the paper's own split (Section 4.1): stars in the 5 x 5 grid nodes around
 *         the point directly, all other stars through the node's Taylor series.  The truncation
 *         error is bounded by rho^(order+1), rho = 0.283; with the default
 *         order 31 it is below FP64 rounding, so the root sets are the same within the parity
 *         tolerance.  The Aberth sum over the other roots stays direct in both modes.             */
enum { MLCC_STAR_SUMS_DIRECT = 0, MLCC_STAR_SUMS_FMM = 1 };

/* Kernel regimes of the solver (mlcc_options.regime; how much of the GPU one phase fills).
 * TILED: every iteration of all rows in flight is a few launches over a persistent grid that tiles roots and
 *        sources through shared memory (any N; the path for N >~ 10^3).
 * CHAIN: one CTA owns a sub-chain and runs all its rows and iterations out of shared memory, one launch per call
 *        (fields of up to about 1200 stars; direct star sums, disc fields, FP64 Aberth sum, no trust_predictor).
 * AUTO:  CHAIN where it applies and n_r <= 2400 (all that fits shared memory), else TILED.
 *        The root sets are the same within the parity
 *        tolerance; the bits differ (other summation order).                                              */
enum { MLCC_REGIME_AUTO = 0, MLCC_REGIME_TILED = 1, MLCC_REGIME_CHAIN = 2 };

/* Options of mlcc_critical_curves_ex.  Zero-initialise, or call mlcc_options_default(). */
typedef struct mlcc_options {
    int32_t struct_size;      /* = sizeof(mlcc_options)                                             */
    int32_t num_subchains;    /* sub-chains grown concurrently from their centre rows outwards
                                 (PAPER.md:211-213); 0 = chosen from N and num_phi                  */
    int32_t predictor_order;  /* seeds of a new row: 0 = the previous row's roots;
                                 p >= 1 = polynomial extrapolation through up to p+1 rows of the chain, the
                                 order chosen root by root: terms are added only while they still fall by a
                                 factor two from one order to the next, so a rough or noisy history falls
                                 back towards the previous row's root (result-preserving: only the starting
                                 guess changes); max 8; -1 = library default (8)                     */
    int32_t max_iter_cold;    /* iteration cap of the cold-started centre rows; 0 = max_iter        */
    int64_t phi_index_offset; /* row j has phase phi = 2 pi (j + phi_index_offset) / phi_index_total */
    int64_t phi_index_total;  /* 0 = num_phi (the half-open grid over [0, 2 pi))                     */
    int32_t min_lanes_per_root; /* lower bound on the threads that split one root's sums
                                   (power of two <= 128); 0 = library default                        */
    int32_t aberth_sum_precision; /* arithmetic of the Aberth sum A = sum_{r != k} 1/(z_k - z_r)
                                   (Eq. 17).  A multiplies F in the denominator of the
                                   update, so it steers the convergence rate only: the fixed point
                                   F = 0 and the freeze test do not depend on it (R19).
                                   0 or 64 = FP64 differences with the 20-bit reciprocal seed (the
                                   default: every pair of the iteration is FP64 arithmetic);
                                   32 = double-single FP32 (z = hi + lo, differences exact to
                                   ~2^-23 |z_k - z_r|, packed f32x2 instructions; tiled regime only;
                                   about 9 % faster at N = 10^4).  Star sums (F, F') are FP64 in both. */
    int32_t star_sum_mode;    /* MLCC_STAR_SUMS_DIRECT (default) or MLCC_STAR_SUMS_FMM               */
    int32_t fmm_order;        /* Taylor order of the node series (1..63); 0 = 31                     */
    int32_t fmm_stars_per_node; /* mean stars per grid node (the grid has ~N / this many nodes);
                                   0 = 4                                                             */
    int32_t trust_predictor;  /* 0 (default): the first iteration of every row evaluates the Aberth sum for
                                 every root.  1: a row whose seeds come from the predictor at its full
                                 order (predictor_order >= 1) starts with Newton steps (no Aberth sum);
                                 a step below skip_aberth_sum_below is applied and confirmed as usual, a
                                 larger one is discarded and that root gets a full Aberth iteration from
                                 its seed instead.  Cold rows, low-order rows and every root whose
                                 prediction was off keep Eq. 17 as printed; the fixed point F = 0 and the
                                 freeze test are the same (reading R30).  Needs
                                 skip_aberth_sum_below >= 0.                                         */
    /* Smooth-sheet polynomial (rectangular microlens field, PAPER.md:197-205 and Appendix B).  With
       H(u) = sum_{n=0}^{d} sheet_poly[n] u^n (REAL coefficients) the lens equation becomes
         w = (1-kappa_s) z + gamma conj(z) - conj( sum_i m_i/(z - z_i) + H(z) ),
       so F = gamma + S2 - H'(z) - (1-kappa_s) e^{-i phi}, F' = -2 S3 - H''(z), and every row has
       2N + d - 1 roots (d >= 2).  mlcc_rect_sheet fills the coefficients from
       Eq. B2; the caller adds its gamma_shift to gamma.  NULL / 0 = the infinite sheet of a disc. */
    const double *sheet_poly; /* HOST pointer, [sheet_poly_n]; the last coefficient must be non-zero  */
    int32_t sheet_poly_n;     /* d + 1, at most 512; 0 = none                                        */
    int32_t regime;           /* MLCC_REGIME_AUTO (default), _TILED or _CHAIN: see the enum above                    */
    double seed_radius;       /* the d - 1 extra cold seeds are spread evenly on the circle of this
                                 radius about the origin; must be > 0 when d >= 2 and
                                 init_roots is NULL                                                   */
    double skip_aberth_sum_below; /* A root whose step |dz| was below this (but not below tol) is iterated
                                 the next time with the Newton step dz = F/F' (Eq. 17 without the term
                                 F (2 S1 - A)): that iteration only confirms |dz| < tol, and the term,
                                 which multiplies F ~ F' dz in the denominator, cannot move the step by
                                 more than |dz|^2 |2 S1 - A| (reading R27).  The first iteration of every row always has A, and so
                                 has every root whose last step was larger.  0 = library default
                                 (1e-8 in the chain regime and, in the tiled regime, for N >= 512: smaller
                                 fields are launch bound there and the extra launch costs more than it
                                 saves, unless trust_predictor is set); negative = never skip.       */
} mlcc_options;

/* Counters of one mlcc_critical_curves_ex call (host struct, filled on return). */
typedef struct mlcc_stats {
    int64_t root_iterations;   /* sum over all Aberth iterations of the number of unfrozen roots updated */
    int64_t star_pairs;        /* (root, star) pair evaluations  = root_iterations * N                  */
    int64_t root_pairs;        /* (root, root) pair evaluations: (2N - 1) per root-iteration that had the
                                  Aberth sum (see mlcc_options.skip_aberth_sum_below)                    */
    int64_t kernel_launches;   /* kernels launched by the call (chain regime: 2)                        */
    int32_t total_iterations;  /* Aberth iterations summed over steps (one step = all chains advance 1 row);
                                  chain regime: those of the sub-chain that ran the most (the critical path)  */
    int32_t steps;             /* steps taken (cold step included)                                      */
    int32_t subchains;         /* sub-chains used                                                       */
    int32_t predictor_order;   /* predictor order used                                                  */
    int32_t unconverged_rows;  /* rows with out_unconverged > 0                                         */
    int32_t degenerate_roots;  /* NaN/Inf steps seen                                                    */
    float   solve_ms;          /* device time of the call's kernels, CUDA events on `stream`            */
    int32_t aberth_sum_precision; /* 32 or 64: the Aberth-sum arithmetic used                           */
    int32_t regime;            /* MLCC_REGIME_TILED or MLCC_REGIME_CHAIN: the regime used               */
    int32_t reserved_;
} mlcc_stats;

int         mlcc_version(void);                 /* major*10000 + minor*100 + patch                       */
const char *mlcc_status_string(int status);     /* static string                                         */
const char *mlcc_last_error(void);              /* text of the calling thread's last failure ("" if none) */
void        mlcc_options_default(mlcc_options *opt /*host*/);

/* a0  Star field (Eq. 9, with A_star = pi R^2).
 * N stars uniform in the disk of radius R = sqrt(N / kappa_star) around the origin, masses from
 * `mass_model`, divided by their sample mean so that sum m_i = N (theta_star is the Einstein
 * radius of the mean mass).  Counter-based Philox4x32-10 keyed by `seed`; the recipe is in
 * DESIGN.md "Input recipe" and the same seed gives the same field on every call.
 *   mass_params (host, may be NULL = defaults):
 *     MLCC_MASS_EQUAL: ignored.
 *     MLCC_MASS_POWER_LAW: {m_lo, m_hi, alpha}, dN/dm ~ m^-alpha (default 0.08, 1, 2.35).
 *     MLCC_MASS_BROKEN_POWER_LAW: {m0, m1, m2, m3, alpha1, alpha2, alpha3}, continuous at m1, m2
 *       (default 0.01, 0.08, 0.5, 1.5, 0.3, 1.3, 2.3).
 *   star_xy [N][2], masses [N]: device, written.  out_radius: host, may be NULL.
 * Synchronises `stream`.  Errors: INVALID_ARG (N < 1, kappa_star <= 0, bad model/params), CUDA.  */
int mlcc_star_field(uint64_t seed, int64_t N, double kappa_star, int mass_model,
                    const double *mass_params, double *star_xy, double *masses,
                    double *out_radius, void *stream);

/* a0 for the rectangular field of Section 4.2 (Appendix A at :386: stars in the
 * rectangle with corner c = c1 + i c2, sides 2 c1 x 2 c2).  Same masses and seed recipe as
 * mlcc_star_field; Eq. 9 with A_star = 4 c1 c2 and sum m_i = N fixes
 * c2 = sqrt(pi N / (4 kappa_star aspect)), c1 = aspect c2  (aspect = c1/c2 > 0).  Star i sits at
 * (c1 x, c2 y) with x, y uniform in [-1, 1) from Philox counter (i, 0, 0).  Feed c1, c2 to
 * mlcc_rect_sheet for the matching smooth sheet.
 *   star_xy [N][2], masses [N]: device, written.  out_corner [2]: host, may be NULL, gets {c1, c2}.
 * Synchronises `stream`.  Errors: INVALID_ARG (also aspect <= 0 or non-finite), CUDA.              */
int mlcc_star_field_rect(uint64_t seed, int64_t N, double kappa_star, double aspect, int mass_model,
                         const double *mass_params, double *star_xy, double *masses,
                         double *out_corner, void *stream);

/* a1-a6  Critical curves (PAPER.md:128 Eq. 15, :159 Eq. 17, :170 Eq. 19, :176-182, :211-213).
 * For each row j of the grid phi_j = 2 pi j / num_phi finds all 2N roots of F(z, phi_j) by the
 * Aberth–Ehrlich iteration evaluated from the rational form (O(N) star sums and an O(N) sum over
 * the other roots per root and iteration), every root frozen once its step |dz| < tol, roots of
 * one row seeding the next along each chain.
 *   star_xy [N][2], masses [N]: device, read.
 *   out_roots [num_phi][2N][2]: device, written.  Row j is the root SET of phi_j; the column
 *     order is continuous along a sub-chain but otherwise unspecified.  (With a sheet polynomial,
 *     mlcc_options.sheet_poly, every array documented as [..][2N] is [..][mlcc_num_roots()].)
 * Default options and the default stream; returns after the work has finished.
 * Errors: INVALID_ARG, CUDA, NOMEM, NOT_CONVERGED, DEGENERATE (outputs are written in the last two). */
int mlcc_critical_curves(const double *star_xy, const double *masses, int64_t N,
                         double kappa_s, double gamma, int64_t num_phi, double tol,
                         int32_t max_iter, double *out_roots);

/* As above with options, an initial guess, per-row diagnostics and a stream.
 *   opt: host, NULL = defaults.
 *   init_roots [2N][2]: device or NULL.  Starting approximations of every cold-started centre row
 *     instead of the paper's z_i +/- 1.
 *   out_iters [num_phi], out_unconverged [num_phi]: device int32 or NULL.  Iterations spent on the
 *     row; roots of the row still unfrozen at max_iter.
 *   out_stats: host or NULL.                                                                     */
int mlcc_critical_curves_ex(const double *star_xy, const double *masses, int64_t N,
                            double kappa_s, double gamma, int64_t num_phi, double tol,
                            int32_t max_iter, double *out_roots,
                            const mlcc_options *opt, const double *init_roots,
                            int32_t *out_iters, int32_t *out_unconverged,
                            mlcc_stats *out_stats, void *stream);

/* a1-a7 fused: critical curves and their caustic points in one pass.  Same as
 * mlcc_critical_curves_ex, and out_caustics [num_phi][2N][2] (device, written, may not alias
 * out_roots) receives w(z) of Eq. 12 for every root.  The Aberth kernel carries
 * Sm = sum_i m_i/(z - z_i) beside the star sums it needs anyway, and writes
 * w(z - dz) from Sm(z - dz) = Sm + dz S2 + dz^2 S3 + O(dz^3 S4): exact to rounding for a frozen
 * root (|dz| < tol).  A root still unfrozen at max_iter gets the caustic point of its last
 * iterate to that order.  Errors: as mlcc_critical_curves_ex.                                   */
int mlcc_curves_and_caustics(const double *star_xy, const double *masses, int64_t N,
                             double kappa_s, double gamma, int64_t num_phi, double tol,
                             int32_t max_iter, double *out_roots, double *out_caustics,
                             const mlcc_options *opt, const double *init_roots,
                             int32_t *out_iters, int32_t *out_unconverged,
                             mlcc_stats *out_stats, void *stream);

/* a7  Caustic mapping (Eq. 12 at :114): w_p = lens equation at points[p].
 *   points [P][2]: device, read.  out_caustics [P][2]: device, written (may not alias points).
 * Asynchronous on `stream` (no device status to read back).  P = 0 is a no-op.
 * Errors: INVALID_ARG, CUDA.                                                                     */
int mlcc_caustics(const double *star_xy, const double *masses, int64_t N, double kappa_s,
                  double gamma, const double *points, int64_t P, double *out_caustics,
                  void *stream);

/* a2 on its own  The four star sums at arbitrary points (Eq. 15 at PAPER.md:128, Eq. 19 at :170,
 * Eq. 12 at :114):  S1 = sum 1/(z-z_i), S2 = sum m_i/(z-z_i)^2, S3 = sum m_i/(z-z_i)^3,
 * Sm = sum m_i/(z-z_i), so that F = gamma + S2 - (1-kappa_s) e^{-i phi}, F' = -2 S3,
 * w = (1-kappa_s) z + gamma conj(z) - conj(Sm).  `mode` is MLCC_STAR_SUMS_DIRECT or
 * MLCC_STAR_SUMS_FMM (`fmm_order`, `fmm_stars_per_node` as in mlcc_options; 0 = defaults).
 *   points [P][2]: device, read.
 *   out_sums [P][8]: device, written: Re S1, Im S1, Re S2, Im S2, Re S3, Im S3, Re Sm, Im Sm.
 * A point that coincides with a star gives non-finite sums.  Asynchronous on `stream`.
 * Errors: INVALID_ARG, CUDA, NOMEM.                                                              */
int mlcc_star_sums(const double *star_xy, const double *masses, int64_t N, const double *points,
                   int64_t P, int mode, int fmm_order, int fmm_stars_per_node, double *out_sums,
                   void *stream);

/* a8  Root-set matching validator (BASELINE.json north_star: "root sets per phase are compared
 * after optimal nearest-neighbour matching").  For each of S sets, every a_i is paired with its
 * nearest b_j (uniform-grid search).  If that map is a bijection it is the matching that
 * minimises every pair's distance, hence also the maximum distance.
 *   a, b [S][n][2]: device, read.
 *   out_max_err [S]: device, max_i |a_i - b_j(i)| (inf if a set holds a non-finite value).
 *   out_bijective [S]: device int32, 1 iff j(.) is a bijection and every pair satisfies
 *     |a_i - b_j(i)| <= rel_tol (1 + |b_j(i)|).
 * Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA, NOMEM.                                   */
int mlcc_match_root_sets(const double *a, const double *b, int64_t S, int64_t n, double rel_tol,
                         double *out_max_err, int32_t *out_bijective, void *stream);

/* a8 for callers that may not allocate device memory (code under CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): the same matching as mlcc_match_root_sets, same arguments, same outputs, but the call
 * allocates and frees NOTHING (no cudaMalloc, cudaMallocAsync, cudaFree, no allocating library routine).  Its
 * bins live in a static device array of 4 MiB that every GPU loading the library holds until the process exits.
 *   Limit: n <= 8192 points per set; a larger n returns MLCC_ERR_INVALID_ARG (use mlcc_match_root_sets).
 *   Every call on a device shares that array and finds the previous call's contents in it (the kernel clears what
 *   it needs at zero itself).  Calls that OVERLAP on the GPU (different streams) race on it: keep the calls of one
 *   device on one stream, or order them with events.
 * Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA.                                                       */
int mlcc_match_root_sets_noalloc(const double *a, const double *b, int64_t S, int64_t n, double rel_tol,
                                 double *out_max_err, int32_t *out_bijective, void *stream);

/* a8, invariants  Completeness certificate of the root sets (BASELINE.json
 * north_star: "exactly the paper's degree of distinct roots per phase").  P(z; phi) =
 * F(z, phi) prod_i (z - z_i)^2 has degree 2N and leading coefficient -c(phi),
 * c = (1 - kappa_s) e^{-i phi} - gamma; its next two coefficients give Vieta's sums
 *   sum_k z_k = 2 sum_i z_i,      sum_k z_k^2 = 2 sum_i z_i^2 + 2 (sum_i m_i) / c(phi),
 * which hold for the full set of 2N roots and fail by the displacement if a root is duplicated,
 * missing or misplaced.  O(2N) per row, no second solve needed.  Disc fields only (no sheet_poly).
 *   roots [num_phi][2N][2]: device, read; row j has phase 2 pi (j + phi_index_offset) / phi_index_total
 *   (phi_index_total = 0: num_phi).
 *   out_e1 [num_phi]: device, |sum z_k - 2 sum z_i| / sum |z_k|.
 *   out_e2 [num_phi]: device, |sum z_k^2 - 2 sum z_i^2 - 2 M / c| / sum |z_k|^2.
 * Converged fp64 root sets give values of order 1e-14 (1e-12 is a safe threshold); a duplicated root
 * gives |z_a - z_b| / sum |z_k|.  Sums in a fixed order: the same bits on every run.
 * Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA, NOMEM.                                    */
int mlcc_vieta_residuals(const double *star_xy, const double *masses, int64_t N, double kappa_s,
                         double gamma, const double *roots, int64_t num_phi,
                         int64_t phi_index_offset, int64_t phi_index_total,
                         double *out_e1, double *out_e2, void *stream);

/* a8, invariants  det J certificate of stored roots (BASELINE.json north_star: "|det J| <= 1e-10 at every root";
 * Eq. C1 first line; the bound of C3).  One pass of the star sums at every point:
 *   F = gamma + S2 - (1 - kappa_s) e^{-i phi}  (Eq. 15),  F' = -2 S3  (Eq. 19),
 *   1/mu = det J = (1 - kappa_s)^2 - |gamma + S2|^2,      newton = |F| / |F'|,
 * newton being, to first order, the distance from the point to the exact root of F.  The plain 1e-10 of
 * BASELINE.json is below what fp64 can represent once |F'| >~ 1e4 (a root 0.03 theta_star from a star, N >~ 2000:
 * SURVEY.md 0.2), so the certificate is scale-aware:
 *   bound_k = 1e-10 + 4 (1 - kappa_s) |F'(z_k)| 2^-52 (1 + |z_k|)          (App. C linearised; R16).
 *   points [num_phi][n][2]: device, read; row j has phase 2 pi (j + phi_index_offset) / phi_index_total
 *     (phi_index_total = 0: num_phi).  n is free (2N for the root sets of a disc field).
 *   out_residuals [num_phi][n][6]: device or NULL, written: Re F, Im F, Re F', Im F', 1/mu, newton.
 *   out_row_newton [num_phi]: device, written: max_k newton.
 *   out_row_detj [num_phi]: device, written: max_k |1/mu_k| / bound_k  (<= 1 certifies the row).
 * A point on a star or a non-finite point gives +inf in both row outputs.  Disc fields only (no sheet_poly).
 * Cost: N pair evaluations per point (20 FP64 instructions each), i.e. about what one confirming iteration of the
 * solver costs for that point.  Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA, NOMEM.                    */
int mlcc_detj_residuals(const double *star_xy, const double *masses, int64_t N, double kappa_s, double gamma,
                        const double *points, int64_t num_phi, int64_t n,
                        int64_t phi_index_offset, int64_t phi_index_total,
                        double *out_residuals, double *out_row_newton, double *out_row_detj, void *stream);

/* (f) NEXT-4, as far as the crossing map needs it: chain joining (fn. 5 at :217: "the
 * start of one chain is the end of another, with chains joining together until closed loops are
 * formed").  Row s of `rows` holds n points in any column order (the root sets of consecutive
 * phases: out_roots of the calls above, whose column order changes between sub-chains and at the
 * wrap from the last row to row 0).  out_next[s][i] is the column of row (s+1) mod S holding the
 * point nearest to point i of row s: roots move continuously with phi, so on a fine
 * enough grid that point continues the chain.  Ties go to the lowest column.
 *   rows [S][n][2]: device, read.  out_next [S][n]: device int32, written (-1 in a row with a
 *   non-finite value).  out_bijective [S]: device int32, 1 iff i -> out_next[s][i] is a bijection.
 * Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA, NOMEM.                                    */
int mlcc_link_rows(const double *rows, int64_t S, int64_t n, int32_t *out_next,
                   int32_t *out_bijective, void *stream);

/* (f) NEXT-2: number of caustic crossings per source pixel (Section 5.1): the
 * winding number, by Sunday's crossing rule, of the oriented polygons whose vertices are the
 * caustic points of consecutive phases: segment (s, i) runs from caustics[s][i] to
 * caustics[s+1][next[s][i]] (next = NULL: column i continues in column i); with closed != 0 the
 * last row joins row 0.  The caustics are traced clockwise as phi increases, so the
 * count is MINUS the counter-clockwise winding number: 1 inside a simple caustic, 0 far away.
 * Pixel (ix, iy) has its centre at (x0 + (ix + 1/2) pixel, y0 + (iy + 1/2) pixel).
 *   caustics [S][n][2]: device, read (out_caustics of the calls above).  next [S][n]: device int32
 *   or NULL (mlcc_link_rows of the ROOTS: the caustic points cross one another, the roots do not).
 *   out_map [ny][nx]: device int32, written.  Segments with a non-finite end are skipped.
 * A pixel whose centre lies on a segment to rounding may get either neighbour's count.
 * Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA, NOMEM.                                    */
int mlcc_crossing_map(const double *caustics, const int32_t *next, int64_t S, int64_t n, int closed,
                      double x0, double y0, double pixel, int32_t nx, int32_t ny, int32_t *out_map,
                      void *stream);

/* (f) NEXT-4, second part: chains and closed loops ("Every one of the initial n_r roots
 * begins and ends a 'chain' of values from 0 to 2 pi ... sometimes 2 or more chains are needed to fully
 * create a closed critical curve"; fn. 5 at :217: "the start of one chain is the end of another, with
 * chains joining together until closed loops are formed").  Chain k is the one that starts in column
 * k of row 0:  chain_col[0][k] = k,  chain_col[s+1][k] = next[s][chain_col[s][k]].
 *   next [S][n]: device int32, read: mlcc_link_rows of the roots (closed: row S-1 links to row 0).
 *   out_chain_col [S][n]: device int32 or NULL, written: the column of row s that holds chain k.
 *   out_chain_end [n]: device int32, written: next[S-1][chain_col[S-1][k]], the column of row 0 where
 *     chain k arrives after the whole turn of phi, i.e. the chain that continues it.
 *   out_loop_id [n]: device int32, written: the smallest chain index on the cycle of
 *     k -> out_chain_end[k] through k; chains with equal ids form one closed critical curve.
 *   out_num_loops [1]: device int32, written: the number of closed loops.
 * A chain that meets an entry outside [0, n) (a row mlcc_link_rows marked -1) has -1 from there on,
 * out_chain_end = -1 and out_loop_id = -1; so has every chain that does not lie on a cycle (possible
 * only if some row of `next` is not a bijection).  Integer work: results are exact.
 * Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA, NOMEM.                                    */
int mlcc_closed_loops(const int32_t *next, int64_t S, int64_t n, int32_t *out_chain_col,
                      int32_t *out_chain_end, int32_t *out_loop_id, int32_t *out_num_loops,
                      void *stream);

/* Rows put into chain order (the paper's (m+1, n_r) matrix whose column is a chain):
 * out[s][k] = points[s][chain_col[s][k]] (NaN where chain_col is outside [0, n)).  Use it on the roots
 * and on the caustic points alike.  points, out [S][n][2]: device, must not overlap; chain_col [S][n]:
 * device int32 (mlcc_closed_loops).  Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA.         */
int mlcc_order_by_chain(const double *points, const int32_t *chain_col, int64_t S, int64_t n,
                        double *out, void *stream);

/* (f) NEXT-4, third part: distance from every source pixel to the nearest caustic for an expanding
 * source (Section 5.2, Fig. 5 top: "calculated from the map of N_caustic crossings
 * using a Euclidean distance transform").  A pixel is a caustic pixel if one of its 4 neighbours
 * inside the map holds a different count (reading R28);
 *   out_distance[iy][ix] = pixel * min over caustic pixels q of |p - q|  (centre to centre; 0 on a
 *   caustic pixel; +inf if the map has no caustic pixel).  The border of the map is not a caustic
 *   (caption of Fig. 5): a value larger than the pixel's distance to the border is a lower bound only.
 *   crossing_map [ny][nx]: device int32, read (out_map of mlcc_crossing_map, or any integer map).
 *   out_distance [ny][nx]: device double, written.
 *   out_d2 [ny][nx]: device int64 or NULL, written: the squared distance in pixels, exact (-1 for +inf).
 * Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA, NOMEM.                                    */
int mlcc_distance_map(const int32_t *crossing_map, int32_t nx, int32_t ny, double pixel,
                      double *out_distance, int64_t *out_d2, void *stream);

/* The same for a source moving along a direction (Fig. 5 bottom, Fig. 6-7).  The
 * direction is the integer vector (ux, uy), not both zero, |ux|, |uy| <= 2^20 (angle atan2(uy, ux)
 * with the y_1 axis; reading R29).  The ray from the centre of pixel p is followed through
 * the pixel grid exactly, to the point where it first enters the interior of a pixel whose count
 * differs from that of p; out_distance is the distance from the centre of p to that point.  If the
 * ray leaves the map first, out_distance is MINUS the distance to the exit point (a lower bound).
 *   crossing_map [ny][nx]: device int32, read.  out_distance [ny][nx]: device double, written.
 * Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA.                                           */
int mlcc_directional_distance_map(const int32_t *crossing_map, int32_t nx, int32_t ny, double pixel,
                                  int32_t ux, int32_t uy, double *out_distance, void *stream);

/* The statistics of Fig. 6-7: the distribution of the distance to the nearest
 * caustic, per direction of motion (Fig. 6: one call per mlcc_directional_distance_map) and split by
 * "where the source happens to lie in the map of N_caustic crossings" (Fig. 7: `crossing_map` given; for
 * the distance BETWEEN the caustics before and behind a moving source pass the sum of the maps of
 * (ux, uy) and (-ux, -uy)).  Pixel p with a finite distance d >= 0 is counted in bin
 * floor(d / bin_width) if that is < num_bins, in row min(max(crossing_map[p], 0), num_counts - 1)
 * (row 0 when crossing_map is NULL).  Negative values (a ray limited by the border of the map), +inf
 * and NaN are left out and counted in *out_left_out.
 *   distance [num_pixels]: device double, read.  crossing_map [num_pixels]: device int32 or NULL.
 *   out_hist [num_counts][num_bins]: device int64, written.  out_left_out [1]: device int64, written.
 * Integer counts: exact and independent of timing.  Asynchronous on `stream`.
 * Errors: INVALID_ARG (also num_bins * num_counts > 2^26), CUDA.                                    */
int mlcc_distance_histogram(const double *distance, const int32_t *crossing_map, int64_t num_pixels,
                            double bin_width, int32_t num_bins, int32_t num_counts,
                            int64_t *out_hist, int64_t *out_left_out, void *stream);

/* (f) NEXT-3: the rectangular sheet of Appendix B as a polynomial (host-only, no CUDA call).
 * For stars in the rectangle with corner c = c1 + i c2 and smooth compensation kappa_star, Eq. B2
 * truncated at the odd power t and extended to an infinite sheet is
 *   alpha_s(z) = -kappa_star z + kappa_star (1 - 4 theta/pi) conj(z) + H(conj z),  theta = Arg c,
 *   H(u) = -(4 kappa_star/pi) sum_{n = 3,5,..,t} sin((n-1) theta) / (n (n-1)) u^n / |c|^(n-1)
 * (the four logarithm series collected by powers; reading R24), so that Eq. 12 and Eq. 15
 * take the form documented at mlcc_options.sheet_poly with gamma replaced by gamma + *out_gamma_shift,
 * *out_gamma_shift = -kappa_star (1 - 4 theta/pi).
 *   t_in > 0: that truncation power (made odd by adding 1).  t_in = 0: the smallest odd t whose error
 *   bound Eq. B5 is below `eps` for |z| <= |c|/s  (s > 1).  In both cases t is then raised
 *   by 2 until (t-1) theta mod pi is at least 0.1 pi away from 0 and pi, so that the
 *   leading coefficient of H' does not vanish.
 *   out_coef [capacity]: host, receives t + 1 coefficients (even powers and n = 1 are zero).
 * Returns t (> 0), or a negative mlcc_status (bad arguments, capacity < t + 1).                     */
int mlcc_rect_sheet(double kappa_star, double c1, double c2, double s, double eps, int32_t t_in,
                    double *out_coef, int32_t capacity, double *out_gamma_shift);

/* Roots per row for N stars and a sheet polynomial of sheet_poly_n coefficients (0 = none).       */
int64_t mlcc_num_roots(int64_t N, int32_t sheet_poly_n);

/* Host-only planning helper of the phase-continuation driver: splits rows
 * [0, num_phi) into `num_subchains` contiguous sub-chains and returns, per sub-chain c, its
 * first row, its centre row (cold-started) and one past its last row.  num_subchains = 0 asks
 * for the library's choice for this N.  Returns the number of sub-chains written (<= capacity),
 * or a negative mlcc_status on bad arguments.  All pointers host.  No CUDA call is made.        */
int mlcc_plan_subchains(int64_t N, int64_t num_phi, int32_t num_subchains, int32_t capacity,
                        int64_t *first_row, int64_t *centre_row, int64_t *end_row);

/* Host-buffer variants (every pointer is a HOST pointer; the library allocates device memory,
 * copies in, runs the device path above on the default stream, copies out and frees).
 * mlcc_curves_and_caustics_host runs the fused a1..a7 pass (mlcc_curves_and_caustics);
 * out_caustics may be NULL (critical curves only).  If out_roots (and out_caustics) are pinned or
 * registered host memory, the rows of every finished step are copied device -> host on a second
 * stream while the later rows are still being solved (a sub-chain's finished rows are one interval
 * growing at both ends), so the 32 bytes per root cross PCIe under the kernels;
 * pageable outputs are copied once at the end.  The results are the same bits either way.          */
int mlcc_critical_curves_host(const double *star_xy, const double *masses, int64_t N,
                              double kappa_s, double gamma, int64_t num_phi, double tol,
                              int32_t max_iter, double *out_roots);
int mlcc_caustics_host(const double *star_xy, const double *masses, int64_t N, double kappa_s,
                       double gamma, const double *points, int64_t P, double *out_caustics);
int mlcc_curves_and_caustics_host(const double *star_xy, const double *masses, int64_t N,
                                  double kappa_s, double gamma, int64_t num_phi, double tol,
                                  int32_t max_iter, const mlcc_options *opt,
                                  double *out_roots, double *out_caustics, mlcc_stats *out_stats);

#ifdef __cplusplus
}
#endif
#endif /* MLCC_H_ */
