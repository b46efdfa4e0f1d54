// certify.cu — the validator's second invariant: det J and the Newton residual of F
// at every stored root, one pass of the star sums per point.
//
//   F(z, phi)  = gamma + S2 - (1-kappa_s) e^{-i phi},  S2 = sum_i m_i/(z-z_i)^2      (Eq. 15)
//   F'(z)      = -2 S3,                                S3 = sum_i m_i/(z-z_i)^3      (Eq. 19)
//   1/mu = det J = (1-kappa_s)^2 - |gamma + S2|^2                                     (Eq. C1 line 1)
//   newton     = |F| / |F'|: to first order the distance from z to the exact root of F.
// A converged root has |F| at the rounding level of the sum, so 1/mu = -2 (1-kappa_s) Re(F e^{i phi}) - |F|^2 (C1-C3,
// PAPER.md:463-471) is bounded by 2 (1-kappa_s) |F| + |F|^2; with |F| <~ |F'| ulp(z) that is the scale-aware bound
//   |1/mu| <= 1e-10 + 4 (1-kappa_s) |F'| 2^-52 (1 + |z|)                              (R16).
// Per row the kernel also leaves max_k newton and max_k |1/mu_k| / bound_k, so that a caller certifies 10^4 rows by
// reading back 2 x 10^4 numbers.
//
// One thread owns R = 2 points; the stars stream through shared memory; 20 FP64 instructions + 1 MUFU per pair
// (pair_star without S1 and Sm): FP64-pipe bound like the solver's star loop.
#include "star_sums.cuh"

#include <math.h>
#include <vector>

namespace mlcc {
namespace {

constexpr int CBLOCK = 128;
constexpr int CTILE = 1024;
constexpr int CR = 2;

__device__ __forceinline__ void atomic_max_nonneg(double *addr, double v)
{
    // non-negative doubles (and +inf) order like their bit patterns
    atomicMax(reinterpret_cast<unsigned long long *>(addr), (unsigned long long)__double_as_longlong(v));
}

__global__ void __launch_bounds__(CBLOCK) k_residuals(const double2 *__restrict__ stars, const double *__restrict__ masses,
                                                      int N, double gamma, double omk, const double2 *__restrict__ rot,
                                                      const double2 *__restrict__ points, long long P, long long n,
                                                      double *__restrict__ out, double *__restrict__ row_newton,
                                                      double *__restrict__ row_detj)
{
    __shared__ double2 s_xy[CTILE];
    __shared__ double s_m[CTILE];
    const int tid = threadIdx.x;
    const long long n_groups = (P + CBLOCK * CR - 1) / (CBLOCK * CR);
    for (long long g = blockIdx.x; g < n_groups; g += gridDim.x) {
        long long pidx[CR];
        double zx[CR], zy[CR];
        StarAcc acc[CR];
#pragma unroll
        for (int r = 0; r < CR; ++r) {
            pidx[r] = g * (CBLOCK * CR) + r * CBLOCK + tid;
            const double2 z = pidx[r] < P ? points[pidx[r]] : make_double2(0.0, 0.0);
            zx[r] = z.x;
            zy[r] = z.y;
            acc[r] = StarAcc{0, 0, 0, 0, 0, 0, 0, 0};
        }
        for (int base = 0; base < N; base += CTILE) {
            const int cnt = min(CTILE, N - base);
            __syncthreads();
            for (int i = tid; i < cnt; i += CBLOCK) {
                s_xy[i] = stars[base + i];
                s_m[i] = masses[base + i];
            }
            __syncthreads();
#pragma unroll 2
            for (int j = 0; j < cnt; ++j) {
                const double2 s = s_xy[j];
                const double m = s_m[j];
#pragma unroll
                for (int r = 0; r < CR; ++r) pair_star<false, false>(zx[r], zy[r], s, m, acc[r]);
            }
        }
#pragma unroll
        for (int r = 0; r < CR; ++r) {
            const bool valid = pidx[r] < P;
            const long long row = valid ? pidx[r] / n : -1;
            double newton = 0.0, scaled = 0.0;
            if (valid) {
                const double2 e = rot[row];
                const double gx = gamma + acc[r].s2x, gy = 2.0 * acc[r].s2h;   // gamma + S2
                const double fx = gx - e.x, fy = gy - e.y;                       // F
                const double px = -2.0 * acc[r].s3x, py = -2.0 * acc[r].s3y;     // F'
                const double inv_mu = omk * omk - (gx * gx + gy * gy);
                const double fabs_ = hypot(fx, fy), pabs = hypot(px, py);
                newton = fabs_ / pabs;
                const double bound = 1e-10 + 4.0 * omk * pabs * 2.220446049250313e-16 * (1.0 + hypot(zx[r], zy[r]));
                scaled = fabs(inv_mu) / bound;
                if (out) {
                    double *o = out + pidx[r] * 6;
                    o[0] = fx; o[1] = fy; o[2] = px; o[3] = py; o[4] = inv_mu; o[5] = newton;
                }
                if (!(newton == newton) || newton < 0.0) newton = INFINITY;   // NaN must not hide in a max
                if (!(scaled == scaled)) scaled = INFINITY;
            }
            // one atomic per warp and row where the warp's points share a row (the usual case), else one per lane
            const long long row0 = __shfl_sync(0xffffffffu, row, 0);
            if (__all_sync(0xffffffffu, row == row0)) {
                for (int o = 16; o > 0; o >>= 1) {
                    newton = fmax(newton, __shfl_xor_sync(0xffffffffu, newton, o));
                    scaled = fmax(scaled, __shfl_xor_sync(0xffffffffu, scaled, o));
                }
                if ((tid & 31) == 0 && row0 >= 0) {
                    atomic_max_nonneg(&row_newton[row0], newton);
                    atomic_max_nonneg(&row_detj[row0], scaled);
                }
            } else if (valid) {
                atomic_max_nonneg(&row_newton[row], newton);
                atomic_max_nonneg(&row_detj[row], scaled);
            }
        }
    }
}

}  // namespace

int detj_residuals_impl(const double *star_xy, const double *masses, int64_t N, double kappa_s, double gamma,
                        const double *points, int64_t num_phi, int64_t n, int64_t phi_off, int64_t phi_total,
                        double *out_residuals, double *out_row_newton, double *out_row_detj, cudaStream_t stream)
{
    if (!star_xy || !masses) return invalid("null pointer");
    if (N < 1 || N > (1 << 29)) return invalid("N out of range");
    if (num_phi < 0 || n < 1) return invalid("num_phi < 0 or n < 1");
    if (!isfinite(kappa_s) || !isfinite(gamma)) return invalid("kappa_s / gamma not finite");
    if (phi_total < 0 || phi_off < 0) return invalid("phi_index_offset / phi_index_total negative");
    if (num_phi == 0) return MLCC_OK;
    if (!points || !out_row_newton || !out_row_detj) return invalid("null pointer");
    if (phi_total == 0) phi_total = num_phi;
    std::vector<double2> rot((size_t)num_phi);
    const double two_pi = 6.283185307179586476925286766559;
    for (int64_t j = 0; j < num_phi; ++j) {
        const double phi = two_pi * (double)(j + phi_off) / (double)phi_total;
        rot[(size_t)j].x = (1.0 - kappa_s) * cos(phi);
        rot[(size_t)j].y = -(1.0 - kappa_s) * sin(phi);
    }
    Workspace ws(stream);
    double2 *d_rot = nullptr;
    MLCC_CUDA(ws.alloc(&d_rot, (size_t)num_phi));
    // the table leaves a pageable host vector: the copy is done before this returns (staged by the runtime)
    MLCC_CUDA(cudaMemcpyAsync(d_rot, rot.data(), sizeof(double2) * (size_t)num_phi, cudaMemcpyHostToDevice, stream));
    MLCC_CUDA(cudaMemsetAsync(out_row_newton, 0, sizeof(double) * (size_t)num_phi, stream));
    MLCC_CUDA(cudaMemsetAsync(out_row_detj, 0, sizeof(double) * (size_t)num_phi, stream));
    const long long P = (long long)num_phi * n;
    int blocks_per_sm = 0;
    MLCC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, k_residuals, CBLOCK, 0));
    if (blocks_per_sm < 1) blocks_per_sm = 1;
    const long long n_groups = (P + CBLOCK * CR - 1) / (CBLOCK * CR);
    const long long grid_max = (long long)device_sm_count() * blocks_per_sm;
    const int grid = (int)(n_groups < grid_max ? n_groups : grid_max);
    k_residuals<<<grid, CBLOCK, 0, stream>>>(reinterpret_cast<const double2 *>(star_xy), masses, (int)N, gamma,
                                             1.0 - kappa_s, d_rot, reinterpret_cast<const double2 *>(points), P, n,
                                             out_residuals, out_row_newton, out_row_detj);
    MLCC_CUDA(cudaGetLastError());
    return MLCC_OK;
}

}  // namespace mlcc
