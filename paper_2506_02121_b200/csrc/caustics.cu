// caustics.cu — caustic mapping: every critical point through the lens equation.
//
// Eq. 12 with alpha_s = -kappa_star z:
//   w = (1-kappa_s) z + gamma conj(z) - sum_i m_i / (conj(z) - conj(z_i))
// and m/(conj(z)-conj(z_i)) = m (z - z_i)/|z - z_i|^2.
//
// One point per group of T threads (T = 1..32, chosen on the host from P so that small inputs
// still fill the machine); stars stream through shared memory; the T partial sums are combined
// with warp shuffles.
#include "mlcc_common.cuh"

namespace mlcc {
namespace {

constexpr int BLOCK = 256;
constexpr int TILE = 1024;

__global__ void __launch_bounds__(BLOCK) k_caustics(const double2 *__restrict__ stars,
                                                    const double *__restrict__ masses, int N,
                                                    double one_minus_kappa_s, double gamma,
                                                    const double2 *__restrict__ points, long long P,
                                                    double2 *__restrict__ out, int T)
{
    __shared__ double2 s_xy[TILE];
    __shared__ double s_m[TILE];
    const int tid = threadIdx.x;
    const int sub = tid % T;
    const int per_block = BLOCK / T;
    const long long n_groups = (P + per_block - 1) / per_block;
    for (long long g = blockIdx.x; g < n_groups; g += gridDim.x) {
        const long long pidx = g * per_block + tid / T;
        const bool valid = pidx < P;
        double zx = 0.0, zy = 0.0;
        if (valid) {
            const double2 z = points[pidx];
            zx = z.x;
            zy = z.y;
        }
        double ax = 0.0, ay = 0.0;
        for (int base = 0; base < N; base += TILE) {
            const int cnt = min(TILE, N - base);
            __syncthreads();
            for (int i = tid; i < cnt; i += BLOCK) {
                s_xy[i] = stars[base + i];
                s_m[i] = masses[base + i];
            }
            __syncthreads();
            if (valid) {
#pragma unroll 4
                for (int j = sub; j < cnt; j += T) {
                    const double2 s = s_xy[j];
                    const double dx = zx - s.x;
                    const double dy = zy - s.y;
                    const double r2 = fma(dy, dy, fma(dx, dx, 1e-300));   // a point on a star contributes 0
                    const double minv = s_m[j] * rcp_full(r2);
                    ax = fma(dx, minv, ax);
                    ay = fma(dy, minv, ay);
                }
            }
        }
        for (int o = T >> 1; o > 0; o >>= 1) {
            ax += __shfl_xor_sync(0xffffffffu, ax, o);
            ay += __shfl_xor_sync(0xffffffffu, ay, o);
        }
        if (valid && sub == 0) {
            double2 w;
            w.x = fma(one_minus_kappa_s + gamma, zx, -ax);   // (1-kappa_s) x + gamma x - Re sum
            w.y = fma(one_minus_kappa_s - gamma, zy, -ay);   // (1-kappa_s) y - gamma y - Im sum
            out[pidx] = w;
        }
    }
}

}  // namespace

int caustics_impl(const double *star_xy, const double *masses, int64_t N, double kappa_s,
                  double gamma, const double *points, int64_t P, double *out, cudaStream_t stream)
{
    if (!star_xy || !masses) return invalid("null pointer");
    if (N < 1 || N > (1 << 29)) return invalid("N out of range");
    if (P < 0) return invalid("P < 0");
    if (!isfinite(kappa_s) || !isfinite(gamma)) return invalid("kappa_s / gamma not finite");
    if (P == 0) return MLCC_OK;
    if (!points || !out) return invalid("null pointer");
    if (points == out) return invalid("out_caustics aliases points");
    int blocks_per_sm = 0;
    MLCC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, k_caustics, BLOCK, 0));
    if (blocks_per_sm < 1) blocks_per_sm = 1;
    const int grid_max = device_sm_count() * blocks_per_sm;
    int T = 1;
    while (T < 32 && (long long)P * T * 2 <= (long long)grid_max * BLOCK) T <<= 1;
    const long long n_groups = (P + (BLOCK / T) - 1) / (BLOCK / T);
    const int grid = (int)(n_groups < grid_max ? n_groups : grid_max);
    k_caustics<<<grid, BLOCK, 0, stream>>>(reinterpret_cast<const double2 *>(star_xy), masses,
                                           (int)N, 1.0 - kappa_s, gamma,
                                           reinterpret_cast<const double2 *>(points), (long long)P,
                                           reinterpret_cast<double2 *>(out), T);
    MLCC_CUDA(cudaGetLastError());
    return MLCC_OK;
}

}  // namespace mlcc
