// match.cu — root-set matching validator (BASELINE.json north_star).
//
// For each of S sets: every a_i is paired with its nearest b_j.  If i -> j(i) is a bijection,
// it is the perfect matching in which every pair has its least possible distance, so its
// largest distance is the optimum of the bottleneck assignment.
//
// One CTA per set (grid-stride over sets).  b is binned into a uniform G x G grid over its
// bounding box (G^2 ~ n cells) by a counting sort in global scratch; each a_i searches the
// (2r+1)^2 cells around its own, r = 1, 2, ... until the best distance found is <= r * cell size
// (every unsearched point is then farther away), falling back to all of b after r = 4.
#include "mlcc_common.cuh"

namespace mlcc {
namespace {

constexpr int BLOCK = 256;

__device__ __forceinline__ double block_reduce(double v, bool take_max, double *s_buf)
{
    const int tid = threadIdx.x;
    s_buf[tid] = v;
    __syncthreads();
    for (int o = BLOCK / 2; o > 0; o >>= 1) {
        if (tid < o) s_buf[tid] = take_max ? fmax(s_buf[tid], s_buf[tid + o]) : fmin(s_buf[tid], s_buf[tid + o]);
        __syncthreads();
    }
    const double r = s_buf[0];
    __syncthreads();
    return r;
}

__device__ __forceinline__ int cell_coord(double v, double lo, double inv_h, int G)
{
    double c = floor((v - lo) * inv_h);
    if (!(c > 0.0)) c = 0.0;           // also catches NaN
    if (c > (double)(G - 1)) c = (double)(G - 1);
    return (int)c;
}

__global__ void __launch_bounds__(BLOCK) k_match(const double2 *__restrict__ a, const double2 *__restrict__ b,
                                                 long long S, int n, double rel_tol, int G,
                                                 int *scratch, long long scratch_stride,
                                                 double *out_max_err, int *out_bijective,
                                                 long long b_shift, int *out_index)
{
    __shared__ double s_buf[BLOCK];
    __shared__ int s_scan[BLOCK];
    __shared__ int s_flag;
    const int tid = threadIdx.x;
    const int ncell = G * G;
    int *cell_start = scratch + (long long)blockIdx.x * scratch_stride;  // [ncell + 1]
    int *cursor = cell_start + ncell + 1;                                // [ncell]
    int *sorted = cursor + ncell;                                        // [n]
    int *hits = sorted + n;                                              // [n]

    for (long long s = blockIdx.x; s < S; s += gridDim.x) {
        // b_shift = 0: set s of a against set s of b.  b_shift = 1 (chain joining): row s against row (s+1) mod S
        const double2 *as = a + s * n, *bs = b + ((s + b_shift) % S) * n;
        // ---- bounding box of b, finiteness of a and b ----
        double xmin = 1e308, xmax = -1e308, ymin = 1e308, ymax = -1e308, bad = 0.0;
        for (int j = tid; j < n; j += BLOCK) {
            const double2 q = bs[j], q2 = as[j];
            xmin = fmin(xmin, q.x); xmax = fmax(xmax, q.x);
            ymin = fmin(ymin, q.y); ymax = fmax(ymax, q.y);
            if (!(fabs(q.x) <= 1e300) || !(fabs(q.y) <= 1e300) || !(fabs(q2.x) <= 1e300) || !(fabs(q2.y) <= 1e300)) bad = 1.0;
        }
        xmin = block_reduce(xmin, false, s_buf); xmax = block_reduce(xmax, true, s_buf);
        ymin = block_reduce(ymin, false, s_buf); ymax = block_reduce(ymax, true, s_buf);
        bad = block_reduce(bad, true, s_buf);
        if (bad > 0.0) {
            if (tid == 0) { if (out_max_err) out_max_err[s] = INFINITY; out_bijective[s] = 0; }
            if (out_index) for (int i = tid; i < n; i += BLOCK) out_index[s * n + i] = -1;
            continue;
        }
        const double wx = xmax - xmin, wy = ymax - ymin;
        const double hx = wx > 0.0 ? wx / G : 1.0, hy = wy > 0.0 ? wy / G : 1.0;
        const double inv_hx = 1.0 / hx, inv_hy = 1.0 / hy;
        const double hmin = fmin(hx, hy);
        // ---- counting sort of b into cells ----
        for (int c = tid; c <= ncell; c += BLOCK) cell_start[c] = 0;
        for (int j = tid; j < n; j += BLOCK) hits[j] = 0;
        __syncthreads();
        for (int j = tid; j < n; j += BLOCK) {
            const double2 q = bs[j];
            const int c = cell_coord(q.y, ymin, inv_hy, G) * G + cell_coord(q.x, xmin, inv_hx, G);
            atomicAdd(&cell_start[c + 1], 1);
        }
        __syncthreads();
        {   // inclusive scan of cell_start[1..ncell] (block-wide, contiguous chunks)
            const int chunk = (ncell + BLOCK - 1) / BLOCK;
            const int lo = 1 + tid * chunk, hi = min(ncell + 1, lo + chunk);
            int sum = 0;
            for (int c = lo; c < hi; ++c) sum += cell_start[c];
            s_scan[tid] = sum;
            __syncthreads();
            if (tid == 0) {
                int run = 0;
                for (int t = 0; t < BLOCK; ++t) { const int v = s_scan[t]; s_scan[t] = run; run += v; }
            }
            __syncthreads();
            int run = s_scan[tid];
            for (int c = lo; c < hi; ++c) { run += cell_start[c]; cell_start[c] = run; }
            __syncthreads();
        }
        for (int c = tid; c < ncell; c += BLOCK) cursor[c] = cell_start[c];
        __syncthreads();
        for (int j = tid; j < n; j += BLOCK) {
            const double2 q = bs[j];
            const int c = cell_coord(q.y, ymin, inv_hy, G) * G + cell_coord(q.x, xmin, inv_hx, G);
            sorted[atomicAdd(&cursor[c], 1)] = j;
        }
        __syncthreads();
        // ---- nearest b for every a ----
        double max_d2 = 0.0;
        int ok = 1;
        for (int i = tid; i < n; i += BLOCK) {
            const double2 p = as[i];
            const int cx = cell_coord(p.x, xmin, inv_hx, G), cy = cell_coord(p.y, ymin, inv_hy, G);
            double best = INFINITY;
            int bj = -1;
            int r_done = 0;
            for (int r = 1; r <= 4; ++r) {
                // ring r-1 .. r: search cells of the (2r+1)^2 block not in the (2r-1)^2 block (r = 1: all 9)
                for (int yy = cy - r; yy <= cy + r; ++yy) {
                    if (yy < 0 || yy >= G) continue;
                    for (int xx = cx - r; xx <= cx + r; ++xx) {
                        if (xx < 0 || xx >= G) continue;
                        if (r > 1 && abs(yy - cy) < r && abs(xx - cx) < r) continue;
                        const int c = yy * G + xx;
                        for (int t = cell_start[c]; t < cell_start[c + 1]; ++t) {
                            const int j = sorted[t];
                            const double2 q = bs[j];
                            const double dx = p.x - q.x, dy = p.y - q.y;
                            const double d2 = dx * dx + dy * dy;
                            if (d2 < best || (d2 == best && j < bj)) { best = d2; bj = j; }
                        }
                    }
                }
                r_done = r;
                const double reach = r * hmin;
                if (best <= reach * reach) break;
                if (cx - r <= 0 && cy - r <= 0 && cx + r >= G - 1 && cy + r >= G - 1) break;  // whole grid seen
            }
            const double reach = r_done * hmin;
            const bool whole = (cx - r_done <= 0 && cy - r_done <= 0 && cx + r_done >= G - 1 && cy + r_done >= G - 1);
            if (!(best <= reach * reach) && !whole) {   // rare: nothing close, look at everything
                for (int j = 0; j < n; ++j) {
                    const double2 q = bs[j];
                    const double dx = p.x - q.x, dy = p.y - q.y;
                    const double d2 = dx * dx + dy * dy;
                    if (d2 < best || (d2 == best && j < bj)) { best = d2; bj = j; }
                }
            }
            max_d2 = fmax(max_d2, best);
            if (out_index) out_index[s * n + i] = bj;
            if (bj >= 0) {
                atomicAdd(&hits[bj], 1);
                const double2 q = bs[bj];
                const double lim = rel_tol * (1.0 + sqrt(q.x * q.x + q.y * q.y));
                if (!(sqrt(best) <= lim)) ok = 0;
            } else {
                ok = 0;
            }
        }
        max_d2 = block_reduce(max_d2, true, s_buf);
        if (tid == 0) s_flag = 1;
        __syncthreads();
        if (!ok) s_flag = 0;
        __syncthreads();
        for (int j = tid; j < n; j += BLOCK) if (hits[j] != 1) s_flag = 0;
        __syncthreads();
        if (tid == 0) { if (out_max_err) out_max_err[s] = sqrt(max_d2); out_bijective[s] = s_flag; }
        __syncthreads();
    }
}

// The same matching with the bins in SHARED memory (sets of up to ~27 000 points: cell table and sorted indices
// are 8 bytes per point): one CTA of 1024 threads per set, counting sort with shared-memory atomics, block-wide scan
// by warp shuffles, the bijection test by a bit per b_j (n marks on n slots without a repeat cover every slot).
// The global-scratch kernel above stays for larger sets.
constexpr int MBLOCK = 1024;

__device__ __forceinline__ double block_reduce_m(double v, bool take_max, double *s_red /*[33]*/)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int o = 16; o > 0; o >>= 1) {
        const double t = __shfl_xor_sync(0xffffffffu, v, o);
        v = take_max ? fmax(v, t) : fmin(v, t);
    }
    __syncthreads();
    if (lane == 0) s_red[warp] = v;
    __syncthreads();
    if (warp == 0) {
        double w = lane < (int)(blockDim.x >> 5) ? s_red[lane] : v;   // (v: this lane's own warp result, a member of the set)
        for (int o = 16; o > 0; o >>= 1) {
            const double t = __shfl_xor_sync(0xffffffffu, w, o);
            w = take_max ? fmax(w, t) : fmin(w, t);
        }
        if (lane == 0) s_red[32] = w;
    }
    __syncthreads();
    return s_red[32];
}

__global__ void __launch_bounds__(MBLOCK) k_match_smem(const double2 *__restrict__ a, const double2 *__restrict__ b,
                                                       long long S, int n, double rel_tol, int G,
                                                       double *out_max_err, int *out_bijective,
                                                       long long b_shift, int *out_index)
{
    extern __shared__ int s_dyn[];
    __shared__ double s_red[33];
    __shared__ int s_part[MBLOCK / 32 + 1];
    __shared__ int s_flag;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, NTH = blockDim.x, nwarps = NTH >> 5;
    const int ncell = G * G;
    int *cell_start = s_dyn;                       // [ncell + 2]
    int *sorted = cell_start + ncell + 2;          // [n]
    unsigned *mask = reinterpret_cast<unsigned *>(sorted + n);   // [(n + 31) / 32]
    const int n_words = (n + 31) >> 5;

    for (long long s = blockIdx.x; s < S; s += gridDim.x) {
        const double2 *as = a + s * n, *bs = b + ((s + b_shift) % S) * n;
        // ---- bounding box of b, finiteness of a and b ----
        double xmin = 1e308, xmax = -1e308, ymin = 1e308, ymax = -1e308, bad = 0.0;
        for (int j = tid; j < n; j += NTH) {
            const double2 q = bs[j], q2 = as[j];
            xmin = fmin(xmin, q.x); xmax = fmax(xmax, q.x);
            ymin = fmin(ymin, q.y); ymax = fmax(ymax, q.y);
            if (!(fabs(q.x) <= 1e300) || !(fabs(q.y) <= 1e300) || !(fabs(q2.x) <= 1e300) || !(fabs(q2.y) <= 1e300)) bad = 1.0;
        }
        xmin = block_reduce_m(xmin, false, s_red); xmax = block_reduce_m(xmax, true, s_red);
        ymin = block_reduce_m(ymin, false, s_red); ymax = block_reduce_m(ymax, true, s_red);
        bad = block_reduce_m(bad, true, s_red);
        if (bad > 0.0) {
            if (tid == 0) { if (out_max_err) out_max_err[s] = INFINITY; out_bijective[s] = 0; }
            if (out_index) for (int i = tid; i < n; i += NTH) out_index[s * n + i] = -1;
            continue;
        }
        const double wx = xmax - xmin, wy = ymax - ymin;
        const double hx = wx > 0.0 ? wx / G : 1.0, hy = wy > 0.0 ? wy / G : 1.0;
        const double inv_hx = 1.0 / hx, inv_hy = 1.0 / hy;
        const double hmin = fmin(hx, hy);
        // ---- counting sort of b into cells ----
        for (int c = tid; c < ncell + 2; c += NTH) cell_start[c] = 0;
        for (int w = tid; w < n_words; w += NTH) mask[w] = 0u;
        __syncthreads();
        for (int j = tid; j < n; j += NTH) {
            const double2 q = bs[j];
            const int c = cell_coord(q.y, ymin, inv_hy, G) * G + cell_coord(q.x, xmin, inv_hx, G);
            atomicAdd(&cell_start[c + 1], 1);
        }
        __syncthreads();
        {   // inclusive scan of cell_start[1 .. ncell]: cell_start[c + 1] = points in cells 0 .. c
            const int chunk = (ncell + NTH - 1) / NTH;
            const int lo = 1 + tid * chunk, hi = min(ncell + 1, lo + chunk);
            int sum = 0;
            for (int c = lo; c < hi; ++c) sum += cell_start[c];
            int incl = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += t;
            }
            if (lane == 31) s_part[warp] = incl;
            __syncthreads();
            if (warp == 0) {
                const int w = lane < nwarps ? s_part[lane] : 0;
                int wi = w;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int t = __shfl_up_sync(0xffffffffu, wi, o);
                    if (lane >= o) wi += t;
                }
                s_part[lane] = wi - w;
            }
            __syncthreads();
            int run = s_part[warp] + incl - sum;
            for (int c = lo; c < hi; ++c) { run += cell_start[c]; cell_start[c] = run; }
            if (tid == 0) cell_start[ncell + 1] = n;
            __syncthreads();
        }
        // scatter from the back: every insertion into cell c takes slot --cell_start[c + 1]; afterwards
        // cell_start[c + 1] is the FIRST slot of cell c and cell_start[c + 2] one past its last
        for (int j = tid; j < n; j += NTH) {
            const double2 q = bs[j];
            const int c = cell_coord(q.y, ymin, inv_hy, G) * G + cell_coord(q.x, xmin, inv_hx, G);
            sorted[atomicSub(&cell_start[c + 1], 1) - 1] = j;
        }
        __syncthreads();
        // ---- nearest b for every a ----
        double max_d2 = 0.0;
        int ok = 1;
        for (int i = tid; i < n; i += NTH) {
            const double2 p = as[i];
            const int cx = cell_coord(p.x, xmin, inv_hx, G), cy = cell_coord(p.y, ymin, inv_hy, G);
            double best = INFINITY;
            int bj = -1;
            int r_done = 0;
            for (int r = 1; r <= 4; ++r) {
                for (int yy = cy - r; yy <= cy + r; ++yy) {
                    if (yy < 0 || yy >= G) continue;
                    const bool edge_row = abs(yy - cy) == r;
                    // r = 1: the whole 3-cell row is one contiguous range of `sorted`; r > 1: the whole row on the ring's
                    // top and bottom, its two end cells otherwise
                    for (int part = 0; part < 2; ++part) {
                        int xa, xb;
                        if (r == 1 || edge_row) { if (part) break; xa = cx - r; xb = cx + r; }
                        else { xa = xb = part ? cx + r : cx - r; }
                        xa = max(xa, 0);
                        xb = min(xb, G - 1);
                        if (xa > xb) continue;
                        const int t0 = cell_start[yy * G + xa + 1], t1 = cell_start[yy * G + xb + 2];
                        // four candidates per pass: their gathers from b are independent loads in flight together
                        // (the kernel is bound by the latency of these L2 reads); compared in list order as before
                        for (int t = t0; t < t1; t += 4) {
                            int jj[4];
                            double2 qq[4];
#pragma unroll
                            for (int u = 0; u < 4; ++u) jj[u] = sorted[min(t + u, t1 - 1)];
#pragma unroll
                            for (int u = 0; u < 4; ++u) qq[u] = bs[jj[u]];
#pragma unroll
                            for (int u = 0; u < 4; ++u) {
                                if (t + u < t1) {
                                    const int j = jj[u];
                                    const double dx = p.x - qq[u].x, dy = p.y - qq[u].y;
                                    const double d2 = dx * dx + dy * dy;
                                    if (d2 < best || (d2 == best && j < bj)) { best = d2; bj = j; }
                                }
                            }
                        }
                    }
                }
                r_done = r;
                const double reach = r * hmin;
                if (best <= reach * reach) break;
                if (cx - r <= 0 && cy - r <= 0 && cx + r >= G - 1 && cy + r >= G - 1) break;  // whole grid seen
            }
            const double reach = r_done * hmin;
            const bool whole = (cx - r_done <= 0 && cy - r_done <= 0 && cx + r_done >= G - 1 && cy + r_done >= G - 1);
            if (!(best <= reach * reach) && !whole) {   // rare: nothing close, look at everything
                for (int j = 0; j < n; ++j) {
                    const double2 q = bs[j];
                    const double dx = p.x - q.x, dy = p.y - q.y;
                    const double d2 = dx * dx + dy * dy;
                    if (d2 < best || (d2 == best && j < bj)) { best = d2; bj = j; }
                }
            }
            max_d2 = fmax(max_d2, best);
            if (out_index) out_index[s * n + i] = bj;
            if (bj >= 0) {
                const unsigned bit = 1u << (bj & 31);
                if (atomicOr(&mask[bj >> 5], bit) & bit) ok = 0;     // b_j taken twice: not a bijection
                const double2 q = bs[bj];
                const double lim = rel_tol * (1.0 + sqrt(q.x * q.x + q.y * q.y));
                if (!(sqrt(best) <= lim)) ok = 0;
            } else {
                ok = 0;
            }
        }
        max_d2 = block_reduce_m(max_d2, true, s_red);
        const int all_ok = __syncthreads_and(ok);
        if (tid == 0) { if (out_max_err) out_max_err[s] = sqrt(max_d2); out_bijective[s] = all_ok ? 1 : 0; }
        __syncthreads();
    }
    (void)s_flag;
}

// ---- completeness certificate: Vieta's first two sums of every row ----
// P(z; phi) = F(z, phi) prod (z - z_i)^2 has degree 2N and leading coefficient -c(phi); its next two
// coefficients give  sum_k z_k = 2 sum_i z_i  and  sum_k z_k^2 = 2 sum_i z_i^2 + 2 (sum_i m_i)/c(phi).
constexpr int VBLOCK = 256;

// block-wide sum of NQ doubles per thread in a fixed order (the same bits every run); result in every thread
template <int NQ>
__device__ __forceinline__ void block_sum(double (&v)[NQ], double *s_buf /*[NQ][VBLOCK / 32]*/)
{
#pragma unroll
    for (int q = 0; q < NQ; ++q)
        for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0)
#pragma unroll
        for (int q = 0; q < NQ; ++q) s_buf[q * (VBLOCK / 32) + warp] = v[q];
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        double t = 0.0;
        for (int w = 0; w < VBLOCK / 32; ++w) t += s_buf[q * (VBLOCK / 32) + w];
        v[q] = t;
    }
}

// one CTA: star_sums = {Re sum z_i, Im sum z_i, Re sum z_i^2, Im sum z_i^2, sum m_i}
__global__ void __launch_bounds__(VBLOCK) k_vieta_stars(const double2 *__restrict__ stars, const double *__restrict__ masses,
                                                        int N, double *star_sums)
{
    __shared__ double s_buf[5 * (VBLOCK / 32)];
    double v[5] = {0, 0, 0, 0, 0};
    for (int i = threadIdx.x; i < N; i += VBLOCK) {
        const double2 z = stars[i];
        v[0] += z.x; v[1] += z.y;
        v[2] += z.x * z.x - z.y * z.y; v[3] += 2.0 * z.x * z.y;
        v[4] += masses[i];
    }
    block_sum<5>(v, s_buf);
    if (threadIdx.x < 5) star_sums[threadIdx.x] = v[threadIdx.x];
}

// one CTA per row (grid-stride): relative defects of the two sums
__global__ void __launch_bounds__(VBLOCK) k_vieta_rows(const double2 *__restrict__ roots, long long num_phi, int n_r,
                                                       const double *__restrict__ star_sums, double omk, double gamma,
                                                       long long phi_off, long long phi_total,
                                                       double *__restrict__ out_e1, double *__restrict__ out_e2)
{
    __shared__ double s_buf[6 * (VBLOCK / 32)];
    for (long long j = blockIdx.x; j < num_phi; j += gridDim.x) {
        const double2 *row = roots + j * n_r;
        double v[6] = {0, 0, 0, 0, 0, 0};
        for (int k = threadIdx.x; k < n_r; k += VBLOCK) {
            const double2 z = row[k];
            const double a2 = z.x * z.x + z.y * z.y;
            v[0] += z.x; v[1] += z.y;
            v[2] += z.x * z.x - z.y * z.y; v[3] += 2.0 * z.x * z.y;
            v[4] += sqrt(a2); v[5] += a2;
        }
        block_sum<6>(v, s_buf);
        if (threadIdx.x == 0) {
            double sn, cs;
            sincospi(2.0 * (double)(j + phi_off) / (double)phi_total, &sn, &cs);
            const double cx = omk * cs - gamma, cy = -omk * sn;            // c = (1 - kappa_s) e^{-i phi} - gamma
            const double c2 = cx * cx + cy * cy;
            const double qx = 2.0 * star_sums[4] * cx / c2, qy = -2.0 * star_sums[4] * cy / c2;   // 2 M / c
            const double d1x = v[0] - 2.0 * star_sums[0], d1y = v[1] - 2.0 * star_sums[1];
            const double d2x = v[2] - 2.0 * star_sums[2] - qx, d2y = v[3] - 2.0 * star_sums[3] - qy;
            out_e1[j] = sqrt(d1x * d1x + d1y * d1y) / v[4];
            out_e2[j] = sqrt(d2x * d2x + d2y * d2y) / v[5];
        }
        __syncthreads();
    }
}

}  // namespace

int vieta_residuals_impl(const double *star_xy, const double *masses, int64_t N, double kappa_s, double gamma,
                         const double *roots, int64_t num_phi, int64_t phi_index_offset, int64_t phi_index_total,
                         double *out_e1, double *out_e2, cudaStream_t stream)
{
    if (num_phi < 0) return invalid("num_phi < 0");
    if (N < 1 || N > (1 << 28)) return invalid("N out of range");
    if (!isfinite(kappa_s) || !isfinite(gamma)) return invalid("kappa_s / gamma not finite");
    if (num_phi == 0) return MLCC_OK;
    if (!star_xy || !masses || !roots || !out_e1 || !out_e2) return invalid("null pointer");
    const int64_t total = phi_index_total > 0 ? phi_index_total : num_phi;
    Workspace ws(stream);
    double *star_sums = nullptr;
    MLCC_CUDA(ws.alloc(&star_sums, 5));
    k_vieta_stars<<<1, VBLOCK, 0, stream>>>(reinterpret_cast<const double2 *>(star_xy), masses, (int)N, star_sums);
    long long grid = 8ll * device_sm_count();
    if (grid > num_phi) grid = num_phi;
    k_vieta_rows<<<(unsigned)grid, VBLOCK, 0, stream>>>(reinterpret_cast<const double2 *>(roots), (long long)num_phi,
                                                       (int)(2 * N), star_sums, 1.0 - kappa_s, gamma,
                                                       (long long)phi_index_offset, (long long)total, out_e1, out_e2);
    MLCC_CUDA(cudaGetLastError());
    return MLCC_OK;
}

static int match_launch(const double *a, const double *b, int64_t S, int64_t n, double rel_tol,
                        double *out_max_err, int32_t *out_bijective, long long b_shift, int32_t *out_index,
                        cudaStream_t stream);

int match_root_sets_impl(const double *a, const double *b, int64_t S, int64_t n, double rel_tol,
                         double *out_max_err, int32_t *out_bijective, cudaStream_t stream)
{
    if (S < 0) return invalid("S < 0");
    if (n < 1 || n > (1 << 30)) return invalid("n out of range");
    if (!(rel_tol >= 0.0)) return invalid("rel_tol must be >= 0");
    if (S == 0) return MLCC_OK;
    if (!a || !b || !out_max_err || !out_bijective) return invalid("null pointer");
    return match_launch(a, b, S, n, rel_tol, out_max_err, out_bijective, 0, nullptr, stream);
}

// Chain joining (fn. 5 at :217): the successor of every root of row s in row (s+1) mod S.
int link_rows_impl(const double *rows, int64_t S, int64_t n, int32_t *out_next, int32_t *out_bijective,
                   cudaStream_t stream)
{
    if (S < 0) return invalid("S < 0");
    if (n < 1 || n > (1 << 30)) return invalid("n out of range");
    if (S == 0) return MLCC_OK;
    if (!rows || !out_next || !out_bijective) return invalid("null pointer");
    // no distance limit: the flag says only whether every chain has exactly one successor
    return match_launch(rows, rows, S, n, 1.79769313486231570e308, nullptr, out_bijective, 1, out_next, stream);
}

static int match_launch(const double *a, const double *b, int64_t S, int64_t n, double rel_tol,
                        double *out_max_err, int32_t *out_bijective, long long b_shift, int32_t *out_index,
                        cudaStream_t stream)
{
    int G = (int)ceil(sqrt((double)n));
    if (G < 1) G = 1;
    if (G > 2048) G = 2048;
    const long long ncell = (long long)G * G;
    const int sms = device_sm_count();
    // sets whose bins fit shared memory: one 1024-thread CTA per set, everything but the points on chip
    const size_t smem = ((size_t)ncell + 2 + (size_t)n + (size_t)((n + 31) / 32)) * sizeof(int);
    int dev = 0, max_optin = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (smem + 2048 <= (size_t)max_optin) {
        MLCC_CUDA(cudaFuncSetAttribute(k_match_smem, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        // small sets: fewer threads per CTA, more CTAs per SM
        int threads = (int)((n + 31) / 32) * 32;
        if (threads < 64) threads = 64;
        if (threads > MBLOCK) threads = MBLOCK;
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_match_smem, threads, smem) != cudaSuccess || per_sm < 1)
            per_sm = 1;
        long long grid = (long long)per_sm * sms;
        if (grid > S) grid = S;
        k_match_smem<<<(int)grid, threads, smem, stream>>>(reinterpret_cast<const double2 *>(a),
                                                          reinterpret_cast<const double2 *>(b), (long long)S, (int)n,
                                                          rel_tol, G, out_max_err, out_bijective, b_shift, out_index);
        MLCC_CUDA(cudaGetLastError());
        return MLCC_OK;
    }
    const long long stride = (ncell + 1) + ncell + 2 * n;
    // latency-bound CTAs (global-memory counting sort and ring search): as many as stay resident
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_match, BLOCK, 0) != cudaSuccess || per_sm < 1) per_sm = 2;
    long long grid = (long long)per_sm * sms;
    if (grid > S) grid = S;
    Workspace ws(stream);
    int *scratch = nullptr;
    cudaError_t e = ws.alloc(&scratch, (size_t)(stride * grid));
    if (e == cudaErrorMemoryAllocation) {
        cudaGetLastError();
        set_last_error("workspace allocation failed");
        return MLCC_ERR_NOMEM;
    }
    MLCC_CUDA(e);
    k_match<<<(int)grid, BLOCK, 0, stream>>>(reinterpret_cast<const double2 *>(a),
                                            reinterpret_cast<const double2 *>(b), (long long)S, (int)n,
                                            rel_tol, G, scratch, stride, out_max_err, out_bijective, b_shift, out_index);
    MLCC_CUDA(cudaGetLastError());
    return MLCC_OK;
}

// ------------------------------------------------------------------------------------------------
// mlcc_match_root_sets_noalloc: the matcher for callers that may not allocate (code under CUDA graph capture,
// serving loops, harnesses that forbid cudaMalloc).  It runs k_match, the kernel that bins b in GLOBAL scratch, with
// that scratch in the file-scope device array below instead of a per-call allocation: nothing is allocated or freed
// by the call (no cudaMalloc / cudaMallocAsync / cudaFree, no allocating library routine).
//   * Size: MATCH_NOALLOC_INTS ints = 4 MiB, held by every GPU that loads the library until the process exits.
//     A CTA needs (G^2 + 1) + G^2 + 2 n ints, G = ceil(sqrt n); sets of up to MATCH_NOALLOC_MAX_N = 8192 points leave
//     room for >= 31 CTAs.  Larger n is rejected with MLCC_ERR_INVALID_ARG.
//   * In host code the NAME of a __device__ array is a host-side stand-in, not a device address: the address the
//     kernel gets comes from cudaGetSymbolAddress, asked once per device with that device current.
//   * Every call on a device shares the array and finds the previous call's contents in it.  k_match zeroes what it
//     needs at zero (cell counts, hit counts) for every set it handles, so nothing has to be cleared here; but two
//     calls that overlap on the GPU (different streams) RACE on it.  Calls on one stream are ordered and safe.
// ------------------------------------------------------------------------------------------------
constexpr long long MATCH_NOALLOC_INTS = 1ll << 20;
constexpr int MATCH_NOALLOC_MAX_N = 8192;
static __device__ __align__(256) int g_match_scratch[MATCH_NOALLOC_INTS];

int match_root_sets_noalloc_impl(const double *a, const double *b, int64_t S, int64_t n, double rel_tol,
                                 double *out_max_err, int32_t *out_bijective, cudaStream_t stream)
{
    if (S < 0) return invalid("S < 0");
    if (n < 1) return invalid("n < 1");
    if (n > MATCH_NOALLOC_MAX_N)
        return invalid("mlcc_match_root_sets_noalloc: n exceeds 8192 points per set (the static scratch is 4 MiB); "
                       "use mlcc_match_root_sets");
    if (!(rel_tol >= 0.0)) return invalid("rel_tol must be >= 0");
    if (S == 0) return MLCC_OK;
    if (!a || !b || !out_max_err || !out_bijective) return invalid("null pointer");
    // device address of the scratch array, once per device, with that device current
    static int *scratch_of_device[64] = {};
    int dev = 0;
    MLCC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return invalid("device index out of range");
    if (!scratch_of_device[dev]) {
        int *ptr = nullptr;
        MLCC_CUDA(cudaGetSymbolAddress((void **)&ptr, g_match_scratch));
        if (!ptr) return invalid("internal: no device address for the static scratch");
        scratch_of_device[dev] = ptr;
    }
    int *scratch = scratch_of_device[dev];
    int G = (int)ceil(sqrt((double)n));
    if (G < 1) G = 1;
    const long long ncell = (long long)G * G;
    const long long stride = (ncell + 1) + ncell + 2 * n;
    long long grid = MATCH_NOALLOC_INTS / stride;   // CTAs the array has room for (>= 31 by the limit on n)
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_match, BLOCK, 0) != cudaSuccess || per_sm < 1) per_sm = 2;
    const long long resident = (long long)per_sm * device_sm_count();
    if (grid > resident) grid = resident;
    if (grid > S) grid = S;
    if (grid < 1) return invalid("internal: static scratch too small");
    k_match<<<(int)grid, BLOCK, 0, stream>>>(reinterpret_cast<const double2 *>(a), reinterpret_cast<const double2 *>(b),
                                            (long long)S, (int)n, rel_tol, G, scratch, stride, out_max_err,
                                            out_bijective, 0, nullptr);
    MLCC_CUDA(cudaGetLastError());
    return MLCC_OK;
}

}  // namespace mlcc
