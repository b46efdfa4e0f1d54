// crossing.cu — number of caustic crossings per source pixel (§5.1).
//
// "Since the caustics are oriented curves, winding numbers provide the number of caustic crossings ...
// we use a GPU version of Sunday's (2001) algorithm", and fn. 6: "it turns out to be
// computationally faster to loop over the caustic segments and calculate which pixels are affected by a
// given segment".  That is what is done here:
//   * one thread per oriented segment a -> b (row s, column i) -> (row s+1, column next[s][i]);
//   * for every pixel row whose centre line y = py the segment crosses (upward: a.y <= py < b.y, downward:
//     b.y <= py < a.y, Sunday's rule), the crossing abscissa xi; the segment changes the winding number of
//     exactly the pixels of that row whose centre lies left of xi, i.e. columns [0, c): ONE integer atomic
//     on a per-row difference array at column c instead of c updates;
//   * a suffix sum along every row turns the differences into counts.
// Integer atomics commute, so the map is bit-reproducible.  The caustics are traced clockwise
// (PAPER.md:233), so the count is minus the counter-clockwise winding number (reading R21).
#include "mlcc_common.cuh"

namespace mlcc {
namespace {

constexpr int BLOCK = 256;

__global__ void __launch_bounds__(BLOCK) k_cross_scatter(const double2 *__restrict__ caus, const int *__restrict__ next,
                                                         long long S, int n, int closed, double x0, double y0,
                                                         double pixel, int nx, int ny, int *diff)
{
    const long long total = (closed ? S : S - 1) * n;
    const double inv_pixel = 1.0 / pixel;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (long long)gridDim.x * blockDim.x) {
        const long long s = e / n;
        const int i = (int)(e - s * n);
        const long long s1 = (s + 1 == S) ? 0 : s + 1;
        const int j = next ? next[e] : i;
        if (j < 0 || j >= n) continue;
        const double2 a = caus[e], b = caus[s1 * n + j];
        if (!(fabs(a.x) <= 1e300) || !(fabs(a.y) <= 1e300) || !(fabs(b.x) <= 1e300) || !(fabs(b.y) <= 1e300)) continue;
        if (a.y == b.y) continue;   // horizontal: crosses no centre line
        const bool up = a.y < b.y;
        const double lo = up ? a.y : b.y, hi = up ? b.y : a.y;
        // first candidate row: one below the estimate, the exact test decides
        double r0 = ceil((lo - y0) * inv_pixel - 0.5) - 1.0;
        if (r0 < 0.0) r0 = 0.0;
        if (r0 >= (double)ny) continue;
        for (int iy = (int)r0; iy < ny; ++iy) {
            const double py = y0 + ((double)iy + 0.5) * pixel;
            if (py >= hi) break;
            if (py < lo) continue;          // lo <= py < hi: a.y <= py < b.y (up) or b.y <= py < a.y (down)
            const double xi = a.x + (py - a.y) / (b.y - a.y) * (b.x - a.x);
            // c = number of pixel centres of this row with px < xi
            double cf = ceil((xi - x0) * inv_pixel - 0.5);
            if (!(cf > 0.0)) cf = 0.0;
            if (cf > (double)nx) cf = (double)nx;
            int c = (int)cf;
            while (c > 0 && !(x0 + ((double)(c - 1) + 0.5) * pixel < xi)) --c;
            while (c < nx && (x0 + ((double)c + 0.5) * pixel < xi)) ++c;
            if (c > 0) atomicAdd(&diff[(long long)iy * (nx + 1) + c], up ? 1 : -1);
        }
    }
}

// one warp per pixel row: count[ix] = -(sum of diff[c] over c > ix), walking the row from the right
__global__ void __launch_bounds__(BLOCK) k_cross_suffix(const int *__restrict__ diff, int nx, int ny, int *out)
{
    const int row = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31;
    if (row >= ny) return;
    const int *d = diff + (long long)row * (nx + 1);
    int carry = 0;   // sum of diff[c] for c beyond the chunk in hand
    for (int hi = nx; hi > 0; hi -= 32) {
        // lane l handles column ix = hi - 1 - l, which needs diff[ix + 1 .. nx]
        const int ix = hi - 1 - lane;
        int v = ix >= 0 ? d[ix + 1] : 0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, v, o);
            if (lane >= o) v += t;
        }
        if (ix >= 0) out[(long long)row * nx + ix] = -(carry + v);
        carry += __shfl_sync(0xffffffffu, v, 31);
    }
}

}  // namespace

int crossing_map_impl(const double *caustics, const int32_t *next, int64_t S, int64_t n, int closed, double x0,
                      double y0, double pixel, int32_t nx, int32_t ny, int32_t *out_map, cudaStream_t stream)
{
    if (!caustics || !out_map) return invalid("null pointer");
    if (S < 1 || n < 1 || n > (1 << 30)) return invalid("S or n out of range");
    if (nx < 1 || ny < 1 || (long long)nx * ny > (1ll << 31)) return invalid("map size out of range");
    if (!(pixel > 0.0) || !isfinite(pixel) || !isfinite(x0) || !isfinite(y0)) return invalid("x0, y0, pixel");
    Workspace ws(stream);
    int *diff = nullptr;
    const size_t n_diff = (size_t)ny * (nx + 1);
    cudaError_t e = ws.alloc(&diff, n_diff);
    if (e == cudaErrorMemoryAllocation) {
        cudaGetLastError();
        set_last_error("workspace allocation failed");
        return MLCC_ERR_NOMEM;
    }
    MLCC_CUDA(e);
    MLCC_CUDA(cudaMemsetAsync(diff, 0, n_diff * sizeof(int), stream));
    const long long total = (closed ? S : S - 1) * n;
    if (total > 0) {
        long long blocks = (total + BLOCK - 1) / BLOCK;
        const long long cap = 32ll * device_sm_count();
        if (blocks > cap) blocks = cap;
        k_cross_scatter<<<(unsigned)blocks, BLOCK, 0, stream>>>(reinterpret_cast<const double2 *>(caustics), next,
                                                               (long long)S, (int)n, closed, x0, y0, pixel, nx, ny, diff);
    }
    k_cross_suffix<<<(unsigned)(((long long)ny * 32 + BLOCK - 1) / BLOCK), BLOCK, 0, stream>>>(diff, nx, ny, out_map);
    MLCC_CUDA(cudaGetLastError());
    return MLCC_OK;
}

}  // namespace mlcc
