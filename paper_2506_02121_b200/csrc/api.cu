// api.cu — the C-ABI entry points of libmlcc.so (include/mlcc.h) and small host utilities.
#include "mlcc_common.cuh"

#include <math.h>
#include <string.h>

namespace mlcc {

static thread_local std::string g_last_error;

void set_last_error(const std::string &msg) { g_last_error = msg; }

int cuda_fail(cudaError_t e, const char *what, const char *file, int line)
{
    char buf[512];
    snprintf(buf, sizeof buf, "CUDA error %d (%s) at %s:%d: %s", (int)e, cudaGetErrorString(e), file, line, what);
    g_last_error = buf;
    cudaGetLastError();  // clear a non-sticky error
    return e == cudaErrorMemoryAllocation ? MLCC_ERR_NOMEM : MLCC_ERR_CUDA;
}

void keep_pool_memory()
{
    static bool done[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64 || done[dev]) return;
    cudaMemPool_t pool;
    if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
        unsigned long long keep = ~0ull;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    cudaGetLastError();
    done[dev] = true;
}

int device_sm_count()
{
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 1;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) return 1;
    return sms;
}

// implemented in the other translation units
int plan_subchains_host(int64_t, int64_t, int32_t, int32_t, int64_t *, int64_t *, int64_t *);
int critical_curves_impl(const double *, const double *, int64_t, double, double, int64_t, double, int32_t,
                         double *, double *, const mlcc_options *, const double *, int32_t *, int32_t *,
                         mlcc_stats *, cudaStream_t, double *h_roots = nullptr, double *h_caustics = nullptr);
int caustics_impl(const double *, const double *, int64_t, double, double, const double *, int64_t, double *,
                  cudaStream_t);
int star_field_impl(uint64_t, int64_t, double, int, const double *, double, double *, double *, double *, double *,
                    cudaStream_t);
int link_rows_impl(const double *, int64_t, int64_t, int32_t *, int32_t *, cudaStream_t);
int crossing_map_impl(const double *, const int32_t *, int64_t, int64_t, int, double, double, double, int32_t,
                      int32_t, int32_t *, cudaStream_t);
int star_sums_impl(const double *, const double *, int64_t, const double *, int64_t, int, int, int, double *,
                   cudaStream_t);
int closed_loops_impl(const int32_t *, int64_t, int64_t, int32_t *, int32_t *, int32_t *, int32_t *, cudaStream_t);
int order_by_chain_impl(const double *, const int32_t *, int64_t, int64_t, double *, cudaStream_t);
int distance_map_impl(const int32_t *, int32_t, int32_t, double, double *, int64_t *, cudaStream_t);
int directional_distance_map_impl(const int32_t *, int32_t, int32_t, double, int32_t, int32_t, double *,
                                  cudaStream_t);
int distance_histogram_impl(const double *, const int32_t *, int64_t, double, int32_t, int32_t, int64_t *, int64_t *,
                            cudaStream_t);
int match_root_sets_impl(const double *, const double *, int64_t, int64_t, double, double *, int32_t *,
                         cudaStream_t);
int match_root_sets_noalloc_impl(const double *, const double *, int64_t, int64_t, double, double *, int32_t *,
                                 cudaStream_t);
int vieta_residuals_impl(const double *, const double *, int64_t, double, double, const double *, int64_t, int64_t,
                         int64_t, double *, double *, cudaStream_t);

int detj_residuals_impl(const double *, const double *, int64_t, double, double, const double *, int64_t, int64_t,
                        int64_t, int64_t, double *, double *, double *, cudaStream_t);

namespace {

bool host_is_pinned(const void *p)
{
    cudaPointerAttributes a{};
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeHost;
}

struct DeviceBuffer {
    void *p = nullptr;
    ~DeviceBuffer() { if (p) cudaFree(p); }
    cudaError_t alloc(size_t bytes) { return cudaMalloc(&p, bytes ? bytes : 16); }
    template <typename T> T *as() { return static_cast<T *>(p); }
};

}  // namespace
}  // namespace mlcc

using namespace mlcc;

extern "C" {

int mlcc_version(void) { return 100; /* 0.1.0 */ }

const char *mlcc_status_string(int status)
{
    switch (status) {
    case MLCC_OK: return "MLCC_OK";
    case MLCC_ERR_INVALID_ARG: return "MLCC_ERR_INVALID_ARG";
    case MLCC_ERR_CUDA: return "MLCC_ERR_CUDA";
    case MLCC_ERR_NOMEM: return "MLCC_ERR_NOMEM";
    case MLCC_ERR_NOT_CONVERGED: return "MLCC_ERR_NOT_CONVERGED";
    case MLCC_ERR_DEGENERATE: return "MLCC_ERR_DEGENERATE";
    default: return "MLCC_ERR_UNKNOWN";
    }
}

const char *mlcc_last_error(void) { return g_last_error.c_str(); }

void mlcc_options_default(mlcc_options *opt)
{
    if (!opt) return;
    memset(opt, 0, sizeof *opt);
    opt->struct_size = (int32_t)sizeof(mlcc_options);
    opt->num_subchains = 0;
    opt->predictor_order = -1;
    opt->max_iter_cold = 0;
    opt->phi_index_offset = 0;
    opt->phi_index_total = 0;
    opt->min_lanes_per_root = 0;
    opt->aberth_sum_precision = 0;
    opt->star_sum_mode = MLCC_STAR_SUMS_DIRECT;
    opt->fmm_order = 0;
    opt->fmm_stars_per_node = 0;
    opt->trust_predictor = 0;
    opt->sheet_poly = nullptr;
    opt->sheet_poly_n = 0;
    opt->regime = MLCC_REGIME_AUTO;
    opt->seed_radius = 0.0;
    opt->skip_aberth_sum_below = 0.0;
}

int mlcc_star_field(uint64_t seed, int64_t N, double kappa_star, int mass_model, const double *mass_params,
                    double *star_xy, double *masses, double *out_radius, void *stream)
{
    NvtxRange nvtx_("mlcc_star_field");
    return star_field_impl(seed, N, kappa_star, mass_model, mass_params, 0.0, star_xy, masses, out_radius, nullptr,
                           static_cast<cudaStream_t>(stream));
}

int mlcc_star_field_rect(uint64_t seed, int64_t N, double kappa_star, double aspect, int mass_model,
                         const double *mass_params, double *star_xy, double *masses, double *out_corner, void *stream)
{
    NvtxRange nvtx_("mlcc_star_field_rect");
    if (!(aspect > 0.0)) {
        set_last_error("invalid argument: aspect must be positive");
        return MLCC_ERR_INVALID_ARG;
    }
    return star_field_impl(seed, N, kappa_star, mass_model, mass_params, aspect, star_xy, masses, nullptr, out_corner,
                           static_cast<cudaStream_t>(stream));
}

int mlcc_critical_curves(const double *star_xy, const double *masses, int64_t N, double kappa_s, double gamma,
                         int64_t num_phi, double tol, int32_t max_iter, double *out_roots)
{
    NvtxRange nvtx_("mlcc_critical_curves");
    return critical_curves_impl(star_xy, masses, N, kappa_s, gamma, num_phi, tol, max_iter, out_roots, nullptr,
                                nullptr, nullptr, nullptr, nullptr, nullptr, nullptr);
}

int mlcc_critical_curves_ex(const double *star_xy, const double *masses, int64_t N, double kappa_s, double gamma,
                            int64_t num_phi, double tol, int32_t max_iter, double *out_roots,
                            const mlcc_options *opt, const double *init_roots, int32_t *out_iters,
                            int32_t *out_unconverged, mlcc_stats *out_stats, void *stream)
{
    NvtxRange nvtx_("mlcc_critical_curves_ex");
    return critical_curves_impl(star_xy, masses, N, kappa_s, gamma, num_phi, tol, max_iter, out_roots, nullptr,
                                opt, init_roots, out_iters, out_unconverged, out_stats,
                                static_cast<cudaStream_t>(stream));
}

int mlcc_curves_and_caustics(const double *star_xy, const double *masses, int64_t N, double kappa_s, double gamma,
                             int64_t num_phi, double tol, int32_t max_iter, double *out_roots,
                             double *out_caustics, const mlcc_options *opt, const double *init_roots,
                             int32_t *out_iters, int32_t *out_unconverged, mlcc_stats *out_stats, void *stream)
{
    NvtxRange nvtx_("mlcc_curves_and_caustics");
    if (!out_caustics) return invalid("null pointer");
    return critical_curves_impl(star_xy, masses, N, kappa_s, gamma, num_phi, tol, max_iter, out_roots,
                                out_caustics, opt, init_roots, out_iters, out_unconverged, out_stats,
                                static_cast<cudaStream_t>(stream));
}

int mlcc_caustics(const double *star_xy, const double *masses, int64_t N, double kappa_s, double gamma,
                  const double *points, int64_t P, double *out_caustics, void *stream)
{
    NvtxRange nvtx_("mlcc_caustics");
    return caustics_impl(star_xy, masses, N, kappa_s, gamma, points, P, out_caustics,
                         static_cast<cudaStream_t>(stream));
}

int64_t mlcc_num_roots(int64_t N, int32_t sheet_poly_n)
{
    return 2 * N + (sheet_poly_n >= 3 ? sheet_poly_n - 2 : 0);
}

int mlcc_rect_sheet(double kappa_star, double c1, double c2, double s, double eps, int32_t t_in, double *out_coef,
                    int32_t capacity, double *out_gamma_shift)
{
    NvtxRange nvtx_("mlcc_rect_sheet");
    if (!out_coef || !out_gamma_shift) return -invalid("null pointer");
    if (!(kappa_star >= 0.0) || !(c1 > 0.0) || !(c2 > 0.0) || !isfinite(kappa_star + c1 + c2)) return -invalid("kappa_star, c1, c2");
    const double pi = 3.14159265358979323846264338327950288;
    const double cabs = hypot(c1, c2), theta = atan2(c2, c1);
    int t = t_in;
    if (t < 0) return -invalid("t_in < 0");
    if (t == 0) {   // Eq. B5
        if (!(s > 1.0) || !(eps > 0.0)) return -invalid("s must be > 1 and eps > 0");
        t = 1;
        while (kappa_star / pi * 4.0 / (t + 1) * pow(1.0 / s, t + 1) * cabs * (s + 1.0) / (s - 1.0) > eps && t < 2001) t += 2;
    } else if (t % 2 == 0) {
        t += 1;
    }
    for (int guard = 0; guard < 1000; ++guard) {   // keep (t-1) theta away from the multiples of pi
        const double r = fmod((t - 1) * theta, pi);
        if (r >= 0.1 * pi && r <= 0.9 * pi) break;
        t += 2;
    }
    if (t + 1 > capacity || t + 1 > 512) return -invalid("capacity < t + 1 (or t > 511)");
    for (int n = 0; n <= t; ++n) out_coef[n] = 0.0;
    for (int n = 3; n <= t; n += 2)
        out_coef[n] = -(4.0 * kappa_star / pi) * sin((n - 1) * theta) / ((double)n * (n - 1)) / pow(cabs, n - 1);
    *out_gamma_shift = -kappa_star * (1.0 - 4.0 * theta / pi);
    return t;
}

int mlcc_link_rows(const double *rows, int64_t S, int64_t n, int32_t *out_next, int32_t *out_bijective,
                   void *stream)
{
    NvtxRange nvtx_("mlcc_link_rows");
    return link_rows_impl(rows, S, n, out_next, out_bijective, static_cast<cudaStream_t>(stream));
}

int mlcc_crossing_map(const double *caustics, const int32_t *next, int64_t S, int64_t n, int closed, double x0,
                      double y0, double pixel, int32_t nx, int32_t ny, int32_t *out_map, void *stream)
{
    NvtxRange nvtx_("mlcc_crossing_map");
    return crossing_map_impl(caustics, next, S, n, closed, x0, y0, pixel, nx, ny, out_map,
                             static_cast<cudaStream_t>(stream));
}

int mlcc_closed_loops(const int32_t *next, int64_t S, int64_t n, int32_t *out_chain_col, int32_t *out_chain_end,
                      int32_t *out_loop_id, int32_t *out_num_loops, void *stream)
{
    NvtxRange nvtx_("mlcc_closed_loops");
    return closed_loops_impl(next, S, n, out_chain_col, out_chain_end, out_loop_id, out_num_loops,
                             static_cast<cudaStream_t>(stream));
}

int mlcc_order_by_chain(const double *points, const int32_t *chain_col, int64_t S, int64_t n, double *out,
                        void *stream)
{
    NvtxRange nvtx_("mlcc_order_by_chain");
    return order_by_chain_impl(points, chain_col, S, n, out, static_cast<cudaStream_t>(stream));
}

int mlcc_distance_map(const int32_t *crossing_map, int32_t nx, int32_t ny, double pixel, double *out_distance,
                      int64_t *out_d2, void *stream)
{
    NvtxRange nvtx_("mlcc_distance_map");
    return distance_map_impl(crossing_map, nx, ny, pixel, out_distance, out_d2, static_cast<cudaStream_t>(stream));
}

int mlcc_directional_distance_map(const int32_t *crossing_map, int32_t nx, int32_t ny, double pixel, int32_t ux,
                                  int32_t uy, double *out_distance, void *stream)
{
    NvtxRange nvtx_("mlcc_directional_distance_map");
    return directional_distance_map_impl(crossing_map, nx, ny, pixel, ux, uy, out_distance,
                                         static_cast<cudaStream_t>(stream));
}

int mlcc_distance_histogram(const double *distance, const int32_t *crossing_map, int64_t num_pixels, double bin_width,
                            int32_t num_bins, int32_t num_counts, int64_t *out_hist, int64_t *out_left_out, void *stream)
{
    NvtxRange nvtx_("mlcc_distance_histogram");
    return distance_histogram_impl(distance, crossing_map, num_pixels, bin_width, num_bins, num_counts, out_hist,
                                   out_left_out, static_cast<cudaStream_t>(stream));
}

int mlcc_vieta_residuals(const double *star_xy, const double *masses, int64_t N, double kappa_s, double gamma,
                         const double *roots, int64_t num_phi, int64_t phi_index_offset, int64_t phi_index_total,
                         double *out_e1, double *out_e2, void *stream)
{
    NvtxRange nvtx_("mlcc_vieta_residuals");
    return vieta_residuals_impl(star_xy, masses, N, kappa_s, gamma, roots, num_phi, phi_index_offset, phi_index_total,
                                out_e1, out_e2, static_cast<cudaStream_t>(stream));
}

int mlcc_detj_residuals(const double *star_xy, const double *masses, int64_t N, double kappa_s, double gamma,
                        const double *points, int64_t num_phi, int64_t n, int64_t phi_index_offset,
                        int64_t phi_index_total, double *out_residuals, double *out_row_newton, double *out_row_detj,
                        void *stream)
{
    NvtxRange nvtx_("mlcc_detj_residuals");
    return detj_residuals_impl(star_xy, masses, N, kappa_s, gamma, points, num_phi, n, phi_index_offset,
                               phi_index_total, out_residuals, out_row_newton, out_row_detj,
                               static_cast<cudaStream_t>(stream));
}

int mlcc_star_sums(const double *star_xy, const double *masses, int64_t N, const double *points, int64_t P,
                   int mode, int fmm_order, int fmm_stars_per_node, double *out_sums, void *stream)
{
    NvtxRange nvtx_("mlcc_star_sums");
    return star_sums_impl(star_xy, masses, N, points, P, mode, fmm_order, fmm_stars_per_node, out_sums,
                          static_cast<cudaStream_t>(stream));
}

int mlcc_match_root_sets(const double *a, const double *b, int64_t S, int64_t n, double rel_tol,
                         double *out_max_err, int32_t *out_bijective, void *stream)
{
    NvtxRange nvtx_("mlcc_match_root_sets");
    return match_root_sets_impl(a, b, S, n, rel_tol, out_max_err, out_bijective,
                                static_cast<cudaStream_t>(stream));
}

int mlcc_match_root_sets_noalloc(const double *a, const double *b, int64_t S, int64_t n, double rel_tol,
                                 double *out_max_err, int32_t *out_bijective, void *stream)
{
    return match_root_sets_noalloc_impl(a, b, S, n, rel_tol, out_max_err, out_bijective,
                                        static_cast<cudaStream_t>(stream));
}

int mlcc_plan_subchains(int64_t N, int64_t num_phi, int32_t num_subchains, int32_t capacity,
                        int64_t *first_row, int64_t *centre_row, int64_t *end_row)
{
    NvtxRange nvtx_("mlcc_plan_subchains");
    if (!first_row || !centre_row || !end_row) return -MLCC_ERR_INVALID_ARG;
    return plan_subchains_host(N, num_phi, num_subchains, capacity, first_row, centre_row, end_row);
}

int mlcc_curves_and_caustics_host(const double *star_xy, const double *masses, int64_t N, double kappa_s,
                                  double gamma, int64_t num_phi, double tol, int32_t max_iter,
                                  const mlcc_options *opt, double *out_roots, double *out_caustics,
                                  mlcc_stats *out_stats)
{
    NvtxRange nvtx_("mlcc_curves_and_caustics_host");
    if (!star_xy || !masses || !out_roots) return invalid("null pointer");
    if (N < 1 || N > (1 << 28)) return invalid("N out of range");
    if (num_phi < 1) return invalid("num_phi < 1");
    const size_t n_pts = (size_t)num_phi * (size_t)mlcc_num_roots(N, (opt && opt->sheet_poly) ? opt->sheet_poly_n : 0);
    // device copies from the stream-ordered pool (kept cached between calls: mlcc_common.cuh keep_pool_memory; a
    // cudaMalloc / cudaFree pair of 6.4 GB per call cost 0.2-0.3 s at cfg4)
    Workspace hws(nullptr);
    double *d_xy = nullptr, *d_m = nullptr, *d_roots = nullptr, *d_caus = nullptr;
    MLCC_CUDA(hws.alloc(&d_xy, 2 * (size_t)N));
    MLCC_CUDA(hws.alloc(&d_m, (size_t)N));
    MLCC_CUDA(hws.alloc(&d_roots, 2 * n_pts));
    if (out_caustics) MLCC_CUDA(hws.alloc(&d_caus, 2 * n_pts));
    MLCC_CUDA(cudaMemcpyAsync(d_xy, star_xy, sizeof(double) * 2 * (size_t)N, cudaMemcpyHostToDevice, 0));
    MLCC_CUDA(cudaMemcpyAsync(d_m, masses, sizeof(double) * (size_t)N, cudaMemcpyHostToDevice, 0));
    // Pinned (or registered) host outputs receive the finished rows while the solve runs; pageable ones would make
    // every copy block the host thread that feeds the launches, so they are copied once, at the end.
    const bool overlap = host_is_pinned(out_roots) && (!out_caustics || host_is_pinned(out_caustics));
    const int rc = critical_curves_impl(d_xy, d_m, N, kappa_s, gamma, num_phi, tol,
                                        max_iter, d_roots, out_caustics ? d_caus : nullptr,
                                        opt, nullptr, nullptr, nullptr, out_stats, nullptr,
                                        overlap ? out_roots : nullptr, overlap ? out_caustics : nullptr);
    if (rc != MLCC_OK && rc != MLCC_ERR_NOT_CONVERGED && rc != MLCC_ERR_DEGENERATE) return rc;
    const std::string keep = g_last_error;
    if (!overlap) {
        MLCC_CUDA(cudaMemcpyAsync(out_roots, d_roots, sizeof(double) * 2 * n_pts, cudaMemcpyDeviceToHost, 0));
        if (out_caustics)
            MLCC_CUDA(cudaMemcpyAsync(out_caustics, d_caus, sizeof(double) * 2 * n_pts, cudaMemcpyDeviceToHost, 0));
    }
    MLCC_CUDA(cudaStreamSynchronize(0));
    if (rc != MLCC_OK) g_last_error = keep;
    return rc;
}

int mlcc_critical_curves_host(const double *star_xy, const double *masses, int64_t N, double kappa_s,
                              double gamma, int64_t num_phi, double tol, int32_t max_iter, double *out_roots)
{
    NvtxRange nvtx_("mlcc_critical_curves_host");
    return mlcc_curves_and_caustics_host(star_xy, masses, N, kappa_s, gamma, num_phi, tol, max_iter, nullptr,
                                         out_roots, nullptr, nullptr);
}

int mlcc_caustics_host(const double *star_xy, const double *masses, int64_t N, double kappa_s, double gamma,
                       const double *points, int64_t P, double *out_caustics)
{
    NvtxRange nvtx_("mlcc_caustics_host");
    if (!star_xy || !masses) return invalid("null pointer");
    if (N < 1 || N > (1 << 29)) return invalid("N out of range");
    if (P < 0) return invalid("P < 0");
    if (P == 0) return MLCC_OK;
    if (!points || !out_caustics) return invalid("null pointer");
    DeviceBuffer d_xy, d_m, d_pts, d_out;
    MLCC_CUDA(d_xy.alloc(sizeof(double) * 2 * (size_t)N));
    MLCC_CUDA(d_m.alloc(sizeof(double) * (size_t)N));
    MLCC_CUDA(d_pts.alloc(sizeof(double) * 2 * (size_t)P));
    MLCC_CUDA(d_out.alloc(sizeof(double) * 2 * (size_t)P));
    MLCC_CUDA(cudaMemcpyAsync(d_xy.p, star_xy, sizeof(double) * 2 * (size_t)N, cudaMemcpyHostToDevice, 0));
    MLCC_CUDA(cudaMemcpyAsync(d_m.p, masses, sizeof(double) * (size_t)N, cudaMemcpyHostToDevice, 0));
    MLCC_CUDA(cudaMemcpyAsync(d_pts.p, points, sizeof(double) * 2 * (size_t)P, cudaMemcpyHostToDevice, 0));
    const int rc = caustics_impl(d_xy.as<double>(), d_m.as<double>(), N, kappa_s, gamma, d_pts.as<double>(), P,
                                 d_out.as<double>(), nullptr);
    if (rc != MLCC_OK) return rc;
    MLCC_CUDA(cudaMemcpyAsync(out_caustics, d_out.p, sizeof(double) * 2 * (size_t)P, cudaMemcpyDeviceToHost, 0));
    MLCC_CUDA(cudaStreamSynchronize(0));
    return MLCC_OK;
}

}  // extern "C"

