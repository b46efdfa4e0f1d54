// starfield.cu — seeded star-field generator on the device.
//
// Recipe (Eq. 9, with A_star = pi R^2):
//   Philox4x32-10 (Salmon et al. 2011), key = (seed_lo, seed_hi).
//   mass of star i:     counter (i_lo, i_hi, 0, 1), u = u53(r0, r1), inverse CDF of the mass model;
//                       masses are then divided by the sample mean (sum m_i = N).
//   position of star i: counter (i_lo, i_hi, attempt, 0), x = 2 u53(r0,r1) - 1, y = 2 u53(r2,r3) - 1,
//                       first attempt with x*x + y*y < 1 (products and sum rounded separately);
//                       position = R (x, y), R = sqrt(N / kappa_star).
#include "mlcc_common.cuh"

namespace mlcc {
namespace {

constexpr int BLOCK = 256;

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4])
{
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

__device__ __forceinline__ double u53(uint32_t hi, uint32_t lo)
{
    const unsigned long long bits = ((unsigned long long)hi << 32) | (unsigned long long)lo;
    return (double)(bits >> 11) * (1.0 / 9007199254740992.0);
}

struct MassModel {
    int model;
    double lo[3], hi[3], alpha[3];   // segments
    double cum[4], prob[3];
};

__device__ double powerlaw_icdf(double u, double lo, double hi, double alpha)
{
    if (alpha == 1.0) return lo * pow(hi / lo, u);
    const double e = 1.0 - alpha;
    const double a = pow(lo, e), b = pow(hi, e);
    return pow(a + u * (b - a), 1.0 / e);
}

// raw masses + per-block partial sums (fixed tree => same sum on every run)
__global__ void k_masses(MassModel mm, uint32_t k0, uint32_t k1, long long N, double *masses,
                         double *partial)
{
    __shared__ double s_sum[BLOCK];
    double acc = 0.0;
    const long long per_block = (N + gridDim.x - 1) / gridDim.x;
    const long long begin = per_block * blockIdx.x;
    const long long end = begin + per_block < N ? begin + per_block : N;
    for (long long i = begin + threadIdx.x; i < end; i += BLOCK) {
        double m = 1.0;
        if (mm.model != 0) {
            uint32_t r[4];
            philox4x32_10((uint32_t)(i & 0xFFFFFFFFll), (uint32_t)((unsigned long long)i >> 32), 0u, 1u, k0, k1, r);
            const double u = u53(r[0], r[1]);
            if (mm.model == 1) {
                m = powerlaw_icdf(u, mm.lo[0], mm.hi[0], mm.alpha[0]);
            } else {
                const int s = (u < mm.cum[1]) ? 0 : (u < mm.cum[2]) ? 1 : 2;
                const double v = (u - mm.cum[s]) / mm.prob[s];
                m = powerlaw_icdf(v, mm.lo[s], mm.hi[s], mm.alpha[s]);
            }
        }
        masses[i] = m;
        acc += m;
    }
    s_sum[threadIdx.x] = acc;
    __syncthreads();
    for (int o = BLOCK / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) s_sum[threadIdx.x] += s_sum[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = s_sum[0];
}

__global__ void k_mass_total(const double *partial, int n, double *total)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        double s = 0.0;
        for (int i = 0; i < n; ++i) s += partial[i];
        *total = s;
    }
}

// disk: sx = sy = R, rejection from the square.  rectangle: sx = c1, sy = c2, attempt 0 is the star.
__global__ void k_normalise_and_place(uint32_t k0, uint32_t k1, long long N, double sx, double sy, int rect,
                                      const double *total, double *masses, double2 *xy, int *fail)
{
    const double mean = *total / (double)N;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N;
         i += (long long)gridDim.x * blockDim.x) {
        masses[i] = masses[i] / mean;
        double x = 0.0, y = 0.0;
        bool ok = false;
        if (rect) {
            uint32_t r[4];
            philox4x32_10((uint32_t)(i & 0xFFFFFFFFll), (uint32_t)((unsigned long long)i >> 32), 0u, 0u, k0, k1, r);
            x = 2.0 * u53(r[0], r[1]) - 1.0;
            y = 2.0 * u53(r[2], r[3]) - 1.0;
            ok = true;
        }
        for (uint32_t attempt = 0; attempt < 256u && !ok; ++attempt) {
            uint32_t r[4];
            philox4x32_10((uint32_t)(i & 0xFFFFFFFFll), (uint32_t)((unsigned long long)i >> 32), attempt, 0u, k0, k1, r);
            x = 2.0 * u53(r[0], r[1]) - 1.0;
            y = 2.0 * u53(r[2], r[3]) - 1.0;
            ok = __dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y)) < 1.0;
        }
        if (!ok) atomicExch(fail, 1);
        xy[i] = make_double2(__dmul_rn(sx, x), __dmul_rn(sy, y));
    }
}

}  // namespace

// aspect = 0: the disk of mlcc_star_field; aspect > 0: the rectangle of mlcc_star_field_rect (out_corner = {c1, c2})
int star_field_impl(uint64_t seed, int64_t N, double kappa_star, int mass_model,
                    const double *mass_params, double aspect, double *star_xy, double *masses, double *out_radius,
                    double *out_corner, cudaStream_t stream)
{
    if (!(aspect >= 0.0) || !isfinite(aspect)) return invalid("aspect must be positive");
    if (!star_xy || !masses) return invalid("null pointer");
    if (N < 1 || N > (1ll << 29)) return invalid("N out of range");
    if (!(kappa_star > 0.0) || !isfinite(kappa_star)) return invalid("kappa_star must be positive");
    if (mass_model < 0 || mass_model > 2) return invalid("mass_model");
    static const double salpeter[3] = {0.08, 1.0, 2.35};
    static const double kroupa[7] = {0.01, 0.08, 0.5, 1.5, 0.3, 1.3, 2.3};
    MassModel mm{};
    mm.model = mass_model;
    if (mass_model == 1) {
        const double *q = mass_params ? mass_params : salpeter;
        if (!(q[0] > 0.0) || !(q[1] > q[0]) || !isfinite(q[2])) return invalid("power-law mass_params");
        mm.lo[0] = q[0]; mm.hi[0] = q[1]; mm.alpha[0] = q[2];
    } else if (mass_model == 2) {
        const double *q = mass_params ? mass_params : kroupa;
        if (!(q[0] > 0.0) || !(q[1] > q[0]) || !(q[2] > q[1]) || !(q[3] > q[2]))
            return invalid("broken power-law mass_params");
        // dN/dm = A_s m^-alpha_s on segment s, A_1 = 1, continuous at the breaks
        double A[3];
        A[0] = 1.0;
        A[1] = A[0] * pow(q[1], q[5] - q[4]);
        A[2] = A[1] * pow(q[2], q[6] - q[5]);
        double total = 0.0;
        for (int s = 0; s < 3; ++s) {
            mm.lo[s] = q[s]; mm.hi[s] = q[s + 1]; mm.alpha[s] = q[4 + s];
            const double al = mm.alpha[s];
            const double integral = (al == 1.0) ? log(mm.hi[s] / mm.lo[s])
                                                : (pow(mm.hi[s], 1.0 - al) - pow(mm.lo[s], 1.0 - al)) / (1.0 - al);
            mm.prob[s] = A[s] * integral;
            total += mm.prob[s];
        }
        mm.cum[0] = 0.0;
        for (int s = 0; s < 3; ++s) { mm.prob[s] /= total; mm.cum[s + 1] = mm.cum[s] + mm.prob[s]; }
        mm.cum[3] = 1.0;
    }
    const double R = sqrt((double)N / kappa_star);
    // Eq. 9 with A_star = 4 c1 c2 and sum m_i = N
    const double c2 = aspect > 0.0 ? sqrt(3.14159265358979323846 * (double)N / (4.0 * kappa_star * aspect)) : 0.0;
    const double c1 = aspect * c2;
    const uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFull), k1 = (uint32_t)(seed >> 32);

    Workspace ws(stream);
    const int nblk = (int)((N + 4095) / 4096 < 1024 ? (N + 4095) / 4096 : 1024);
    double *partial = nullptr, *total = nullptr;
    int *fail = nullptr;
    MLCC_CUDA(ws.alloc(&partial, (size_t)nblk));
    MLCC_CUDA(ws.alloc(&total, 1));
    MLCC_CUDA(ws.alloc(&fail, 1));
    MLCC_CUDA(cudaMemsetAsync(fail, 0, sizeof(int), stream));
    k_masses<<<nblk, BLOCK, 0, stream>>>(mm, k0, k1, (long long)N, masses, partial);
    k_mass_total<<<1, 32, 0, stream>>>(partial, nblk, total);
    const int grid = (int)((N + BLOCK - 1) / BLOCK < 2048 ? (N + BLOCK - 1) / BLOCK : 2048);
    k_normalise_and_place<<<grid, BLOCK, 0, stream>>>(k0, k1, (long long)N, aspect > 0.0 ? c1 : R, aspect > 0.0 ? c2 : R,
                                                     aspect > 0.0 ? 1 : 0, total, masses,
                                                     reinterpret_cast<double2 *>(star_xy), fail);
    MLCC_CUDA(cudaGetLastError());
    int h_fail = 0;
    MLCC_CUDA(cudaMemcpyAsync(&h_fail, fail, sizeof(int), cudaMemcpyDeviceToHost, stream));
    MLCC_CUDA(cudaStreamSynchronize(stream));
    if (h_fail) {
        set_last_error("internal: rejection sampling exhausted its attempts");
        return MLCC_ERR_CUDA;
    }
    if (out_radius) *out_radius = R;
    if (out_corner && aspect > 0.0) { out_corner[0] = c1; out_corner[1] = c2; }
    return MLCC_OK;
}

}  // namespace mlcc
