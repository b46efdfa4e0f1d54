// fmm.cu — far-field split of the star sums (§4.1): "nearby microlenses are used
// directly, while the distant ones are locally approximated within a node by a Taylor series".
//
// The paper leaves node size and expansion order open ("missing some ideas about the node size and
// requisite expansion order").  Here:
//   * one level: a uniform G x G grid of nodes over the stars' bounding square, G^2 ~ N / stars_per_node;
//   * near = the (2h+1)^2 nodes around the point's node, h = 2;
//   * the node's Taylor coefficients are summed DIRECTLY from every distant star (not translated from
//     node multipoles: the stars are fixed for all phases and iterations, so the series are built once per
//     call at a cost of G^2 N P1 complex multiplications, and no second truncation enters);
//   * order from the geometric bound: a point of the node has |z - c| <= s/sqrt(2), a distant star has
//     |z_i - c| >= (h + 1/2) s, so term l is below rho^l, rho = 0.283; P1 = 32 terms leave < 3e-18.
// Also here: mlcc_star_sums (the four sums at arbitrary points, direct or split), which the parity
// tests use to hold the split against the oracle's straight sums.
#include "star_sums.cuh"

#include <math.h>

namespace mlcc {
namespace {

constexpr int BLOCK = 256;
constexpr int LCHUNK = 8;     // Taylor coefficients one pass of k_fmm_local accumulates per thread

struct Bbox { unsigned long long minx, miny, maxx, maxy; };   // order-preserving keys of the doubles

__device__ __forceinline__ unsigned long long dkey(double v)
{
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    return (b & 0x8000000000000000ull) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double dunkey(unsigned long long k)
{
    const unsigned long long b = (k & 0x8000000000000000ull) ? (k & 0x7fffffffffffffffull) : ~k;
    return __longlong_as_double((long long)b);
}

__global__ void k_fmm_bbox_init(Bbox *bb, int *counts, int n_counts)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) { bb->minx = bb->miny = ~0ull; bb->maxx = bb->maxy = 0ull; }
    for (int j = i; j < n_counts; j += gridDim.x * blockDim.x) counts[j] = 0;
}

__global__ void k_fmm_bbox(const double2 *__restrict__ stars, int N, Bbox *bb)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long a = ~0ull, b = ~0ull, c = 0ull, d = 0ull;
    if (i < N) {
        const double2 z = stars[i];
        a = c = dkey(z.x);
        b = d = dkey(z.y);
    }
    for (int o = 16; o > 0; o >>= 1) {
        a = min(a, __shfl_xor_sync(0xffffffffu, a, o));
        b = min(b, __shfl_xor_sync(0xffffffffu, b, o));
        c = max(c, __shfl_xor_sync(0xffffffffu, c, o));
        d = max(d, __shfl_xor_sync(0xffffffffu, d, o));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMin(&bb->minx, a); atomicMin(&bb->miny, b);
        atomicMax(&bb->maxx, c); atomicMax(&bb->maxy, d);
    }
}

__global__ void k_fmm_geom(const Bbox *bb, int G, FmmGeom *geom)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const double x0 = dunkey(bb->minx), y0 = dunkey(bb->miny), x1 = dunkey(bb->maxx), y1 = dunkey(bb->maxy);
    double side = fmax(x1 - x0, y1 - y0);
    if (!(side > 0.0)) side = 1.0;                 // a single star, or all stars on one point
    const double s = side * (1.0 + 1e-9) / G;      // the largest coordinate falls inside the last node
    geom->x0 = x0 - 0.5 * (s * G - (x1 - x0));     // centre the square on the bounding box
    geom->y0 = y0 - 0.5 * (s * G - (y1 - y0));
    geom->s = s;
    geom->inv_s = 1.0 / s;
}

__device__ __forceinline__ int node_of(const FmmGeom &ge, int G, double2 z)
{
    int ix = (int)((z.x - ge.x0) * ge.inv_s), iy = (int)((z.y - ge.y0) * ge.inv_s);
    ix = min(max(ix, 0), G - 1);
    iy = min(max(iy, 0), G - 1);
    return iy * G + ix;
}

__global__ void k_fmm_count(const double2 *__restrict__ stars, int N, const FmmGeom *geom, int G, int *node,
                            int *counts)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int c = node_of(*geom, G, stars[i]);
    node[i] = c;
    atomicAdd(&counts[c], 1);
}

// exclusive scan of counts[0..n) into start[0..n], one CTA
__global__ void __launch_bounds__(1024) k_fmm_scan(const int *__restrict__ counts, int n, int *start, int *fill)
{
    __shared__ int s_warp[32];
    __shared__ int s_total;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int base = 0;
    for (int c0 = 0; c0 < n; c0 += 1024) {
        const int i = c0 + tid;
        const int v = i < n ? counts[i] : 0;
        int incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            const int w = s_warp[lane];
            int wi = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, wi, o);
                if (lane >= o) wi += t;
            }
            s_warp[lane] = wi - w;
            if (lane == 31) s_total = wi;
        }
        __syncthreads();
        if (i < n) {
            start[i] = base + s_warp[warp] + incl - v;
            fill[i] = 0;
        }
        base += s_total;
        __syncthreads();
    }
    if (tid == 0) start[n] = base;
}

__global__ void k_fmm_scatter(const int *__restrict__ node, int N, const int *__restrict__ start, int *fill,
                              int *order)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int c = node[i];
    order[start[c] + atomicAdd(&fill[c], 1)] = i;
}

// one thread per node: its stars back into their original order (insertion sort of a handful of
// indices), so that the sorted arrays -- and every sum over them -- do not depend on atomic timing
__global__ void k_fmm_order(const int *__restrict__ start, int n_nodes, int *order)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_nodes) return;
    const int a = start[c], b = start[c + 1];
    for (int i = a + 1; i < b; ++i) {
        const int v = order[i];
        int j = i - 1;
        while (j >= a && order[j] > v) { order[j + 1] = order[j]; --j; }
        order[j + 1] = v;
    }
}

__global__ void k_fmm_gather(const double2 *__restrict__ stars, const double *__restrict__ masses,
                             const int *__restrict__ node, const int *__restrict__ order, int N, double2 *sxy,
                             double *sm, int *snode)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const int i = order[j];
    sxy[j] = stars[i];
    sm[j] = masses[i];
    snode[j] = node[i];
}

// Taylor coefficients of one node (one CTA), LCHUNK at a time: thread t sums its share of the distant
// stars, then the CTA adds the shares in a fixed tree.
__global__ void __launch_bounds__(BLOCK) k_fmm_local(FmmGrid g, const int *__restrict__ snode, double2 *Lm,
                                                     double2 *L1)
{
    __shared__ double s_red[BLOCK / 32][4 * LCHUNK];
    const FmmGeom ge = *g.geom;
    const int node = blockIdx.x;
    const int tx = node % g.G, ty = node / g.G;
    const double cx = ge.x0 + (tx + 0.5) * ge.s, cy = ge.y0 + (ty + 0.5) * ge.s;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int l0 = 0; l0 < g.P1; l0 += LCHUNK) {
        double am[2 * LCHUNK], a1[2 * LCHUNK];
#pragma unroll
        for (int q = 0; q < 2 * LCHUNK; ++q) am[q] = a1[q] = 0.0;
        for (int i = tid; i < g.N; i += BLOCK) {
            const int sn = snode[i];
            const int sx = sn % g.G, sy = sn / g.G;
            if (abs(sx - tx) <= g.h && abs(sy - ty) <= g.h) continue;   // near: summed directly at run time
            const double2 z = g.sxy[i];
            const double m = g.sm[i];
            // t = s/(z_i - c)
            const double dx = z.x - cx, dy = z.y - cy;
            const double q = ge.s / (dx * dx + dy * dy);
            const double t_x = dx * q, t_y = -dy * q;
            // w = t^(l0+1): t^8 by squaring, times t for each earlier chunk
            double wx = t_x, wy = t_y;
            if (l0 > 0) {
                double ax = t_x * t_x - t_y * t_y, ay = 2.0 * t_x * t_y;          // t^2
                double bx = ax * ax - ay * ay, by = 2.0 * ax * ay;                // t^4
                ax = bx * bx - by * by; ay = 2.0 * bx * by;                       // t^8
                for (int r = 0; r < l0; r += LCHUNK) {
                    const double nx = wx * ax - wy * ay, ny = wx * ay + wy * ax;
                    wx = nx; wy = ny;
                }
            }
#pragma unroll
            for (int l = 0; l < LCHUNK; ++l) {
                a1[2 * l] -= wx;
                a1[2 * l + 1] -= wy;
                am[2 * l] = fma(-m, wx, am[2 * l]);
                am[2 * l + 1] = fma(-m, wy, am[2 * l + 1]);
                const double nx = wx * t_x - wy * t_y, ny = wx * t_y + wy * t_x;
                wx = nx; wy = ny;
            }
        }
#pragma unroll
        for (int q = 0; q < 2 * LCHUNK; ++q) {
            for (int o = 16; o > 0; o >>= 1) {
                am[q] += __shfl_xor_sync(0xffffffffu, am[q], o);
                a1[q] += __shfl_xor_sync(0xffffffffu, a1[q], o);
            }
        }
        __syncthreads();
        if (lane == 0) {
#pragma unroll
            for (int q = 0; q < 2 * LCHUNK; ++q) { s_red[warp][q] = am[q]; s_red[warp][2 * LCHUNK + q] = a1[q]; }
        }
        __syncthreads();
        if (tid < 4 * LCHUNK) {
            double v = 0.0;
            for (int w = 0; w < BLOCK / 32; ++w) v += s_red[w][tid];
            const int which = tid / (2 * LCHUNK), q = tid % (2 * LCHUNK);
            double2 *dst = (which == 0 ? Lm : L1) + (size_t)node * g.P1 + l0 + q / 2;
            if (q & 1) dst->y = v; else dst->x = v;
        }
    }
}

// the four sums at arbitrary points: one thread per point (split) or T threads per point (direct)
__global__ void k_star_sums_fmm(FmmGrid g, const double2 *__restrict__ points, long long P, double *out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P) return;
    const double2 z = points[i];
    StarAcc a = {0, 0, 0, 0, 0, 0, 0, 0};
    if (!fmm_star_sums(g, z.x, z.y, a)) fmm_direct_all(g, z.x, z.y, a);
    double *o = out + i * 8;
    o[0] = a.s1x; o[1] = a.s1y; o[2] = a.s2x; o[3] = 2.0 * a.s2h; o[4] = a.s3x; o[5] = a.s3y; o[6] = a.smx; o[7] = a.smy;
}

__global__ void __launch_bounds__(BLOCK) k_star_sums_direct(const double2 *__restrict__ stars,
                                                            const double *__restrict__ masses, int N,
                                                            const double2 *__restrict__ points, long long P,
                                                            double *out)
{
    // one warp per point, lanes over stars
    const long long wid = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (wid >= P) return;
    const double2 z = points[wid];
    StarAcc a = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int i = lane; i < N; i += 32) pair_star<true>(z.x, z.y, stars[i], masses[i], a);
    double v[8] = {a.s1x, a.s1y, a.s2x, 2.0 * a.s2h, a.s3x, a.s3y, a.smx, a.smy};
#pragma unroll
    for (int q = 0; q < 8; ++q)
        for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], o);
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < 8; ++q) out[wid * 8 + q] = v[q];
    }
}

}  // namespace

int fmm_build(const double2 *stars, const double *masses, int N, int order, int stars_per_node,
              Workspace &ws, FmmGrid *out, cudaStream_t stream)
{
    if (order < 0 || order > 63) return invalid("fmm_order must be in [0, 63] (0 = default)");
    if (stars_per_node < 0) return invalid("fmm_stars_per_node < 0");
    const int spn = stars_per_node > 0 ? stars_per_node : 4;
    int P1 = order > 0 ? order + 1 : 32;
    P1 = (P1 + LCHUNK - 1) / LCHUNK * LCHUNK;
    int G = (int)ceil(sqrt((double)N / spn));
    if (G < 1) G = 1;
    if (G > 4096) G = 4096;
    const int n_nodes = G * G;
    Bbox *bb = nullptr;
    FmmGeom *geom = nullptr;
    int *counts = nullptr, *start = nullptr, *fill = nullptr, *node = nullptr, *order_idx = nullptr, *snode = nullptr;
    double2 *sxy = nullptr, *Lm = nullptr, *L1 = nullptr;
    double *sm = nullptr;
    cudaError_t e;
    if ((e = ws.alloc(&bb, 1)) != cudaSuccess || (e = ws.alloc(&geom, 1)) != cudaSuccess ||
        (e = ws.alloc(&counts, (size_t)n_nodes)) != cudaSuccess ||
        (e = ws.alloc(&start, (size_t)n_nodes + 1)) != cudaSuccess ||
        (e = ws.alloc(&fill, (size_t)n_nodes)) != cudaSuccess || (e = ws.alloc(&node, (size_t)N)) != cudaSuccess ||
        (e = ws.alloc(&order_idx, (size_t)N)) != cudaSuccess || (e = ws.alloc(&snode, (size_t)N)) != cudaSuccess ||
        (e = ws.alloc(&sxy, (size_t)N)) != cudaSuccess || (e = ws.alloc(&sm, (size_t)N)) != cudaSuccess ||
        (e = ws.alloc(&Lm, (size_t)n_nodes * P1)) != cudaSuccess ||
        (e = ws.alloc(&L1, (size_t)n_nodes * P1)) != cudaSuccess) {
        if (e == cudaErrorMemoryAllocation) {
            cudaGetLastError();
            set_last_error("far-field workspace allocation failed");
            return MLCC_ERR_NOMEM;
        }
        return cuda_fail(e, "cudaMallocAsync", __FILE__, __LINE__);
    }
    const unsigned nb = (unsigned)((N + BLOCK - 1) / BLOCK);
    k_fmm_bbox_init<<<(unsigned)((n_nodes + BLOCK - 1) / BLOCK), BLOCK, 0, stream>>>(bb, counts, n_nodes);
    k_fmm_bbox<<<nb, BLOCK, 0, stream>>>(stars, N, bb);
    k_fmm_geom<<<1, 32, 0, stream>>>(bb, G, geom);
    k_fmm_count<<<nb, BLOCK, 0, stream>>>(stars, N, geom, G, node, counts);
    k_fmm_scan<<<1, 1024, 0, stream>>>(counts, n_nodes, start, fill);
    k_fmm_scatter<<<nb, BLOCK, 0, stream>>>(node, N, start, fill, order_idx);
    k_fmm_order<<<(unsigned)((n_nodes + BLOCK - 1) / BLOCK), BLOCK, 0, stream>>>(start, n_nodes, order_idx);
    k_fmm_gather<<<nb, BLOCK, 0, stream>>>(stars, masses, node, order_idx, N, sxy, sm, snode);
    FmmGrid g;
    g.geom = geom; g.G = G; g.P1 = P1; g.h = 2; g.N = N;
    g.cell_start = start; g.sxy = sxy; g.sm = sm; g.Lm = Lm; g.L1 = L1;
    k_fmm_local<<<(unsigned)n_nodes, BLOCK, 0, stream>>>(g, snode, Lm, L1);
    MLCC_CUDA(cudaGetLastError());
    *out = g;
    return MLCC_OK;
}

int star_sums_impl(const double *star_xy, const double *masses, int64_t N, const double *points, int64_t P,
                   int mode, int order, int stars_per_node, double *out_sums, cudaStream_t stream)
{
    if (!star_xy || !masses) return invalid("null pointer");
    if (N < 1 || N > (1 << 28)) return invalid("N out of range");
    if (P < 0) return invalid("P < 0");
    if (mode != MLCC_STAR_SUMS_DIRECT && mode != MLCC_STAR_SUMS_FMM) return invalid("star_sum_mode");
    if (P == 0) return MLCC_OK;
    if (!points || !out_sums) return invalid("null pointer");
    const double2 *st = reinterpret_cast<const double2 *>(star_xy);
    const double2 *pt = reinterpret_cast<const double2 *>(points);
    if (mode == MLCC_STAR_SUMS_DIRECT) {
        const long long threads = (long long)P * 32;
        k_star_sums_direct<<<(unsigned)((threads + BLOCK - 1) / BLOCK), BLOCK, 0, stream>>>(st, masses, (int)N, pt,
                                                                                           (long long)P, out_sums);
        MLCC_CUDA(cudaGetLastError());
        return MLCC_OK;
    }
    Workspace ws(stream);
    FmmGrid g;
    const int rc = fmm_build(st, masses, (int)N, order, stars_per_node, ws, &g, stream);
    if (rc != MLCC_OK) return rc;
    k_star_sums_fmm<<<(unsigned)((P + 127) / 128), 128, 0, stream>>>(g, pt, (long long)P, out_sums);
    MLCC_CUDA(cudaGetLastError());
    return MLCC_OK;   // the workspace is released in stream order after the kernels
}

}  // namespace mlcc
