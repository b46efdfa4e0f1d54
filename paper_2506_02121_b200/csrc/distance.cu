// distance.cu — distance from every source pixel to the nearest caustic (second part;
// PAPER.md:247, Section 5.2, Fig. 5), computed from the map of the number of caustic crossings.
//
// Expanding source (Fig. 5 top): "calculated from the map of N_caustic crossings using a Euclidean distance
// transform".  A pixel is a caustic pixel if one of its 4 neighbours inside the map holds another count
// (reading R28); the result is pixel * min over caustic pixels q of |p - q|.  Exact, separable:
//   k_edt_columns: g[y][x] = distance along the column to the nearest caustic pixel (one thread per column, an
//                  upward and a downward sweep, loads and stores coalesced over x);
//   k_edt_rows:    d2[y][x] = min over x' of (x - x')^2 + g[y][x']^2, scanning outwards from x and stopping as
//                  soon as (x - x')^2 alone reaches the best value so far: O(distance) work per pixel, in integers.
//
// Moving source (Fig. 5 bottom): the direction is an integer vector u (reading R29); the ray from the
// centre of p is walked through the pixel grid exactly (coordinates doubled: centres even, pixel borders odd;
// border parameters (2 i + 1)/|u| compared by cross-multiplication), to the point where it first enters a pixel
// with another count.  A ray through a pixel corner steps diagonally.  If the ray leaves the map first the result
// is minus the distance to the exit point (the caption of Fig. 5: the border is not a caustic).
#include "mlcc_common.cuh"

namespace mlcc {
namespace {

constexpr int BLOCK = 256;
constexpr int G_INF = 1 << 30;   // "no caustic pixel in this column"; its square still fits in 64 bits

__device__ __forceinline__ bool caustic_pixel(const int *__restrict__ map, int nx, int ny, int x, int y)
{
    const int v = map[(long long)y * nx + x];
    if (x > 0 && map[(long long)y * nx + x - 1] != v) return true;
    if (x + 1 < nx && map[(long long)y * nx + x + 1] != v) return true;
    if (y > 0 && map[(long long)(y - 1) * nx + x] != v) return true;
    if (y + 1 < ny && map[(long long)(y + 1) * nx + x] != v) return true;
    return false;
}

__global__ void __launch_bounds__(BLOCK) k_edt_columns(const int *__restrict__ map, int nx, int ny, int *__restrict__ g)
{
    const int x = blockIdx.x * BLOCK + threadIdx.x;
    if (x >= nx) return;
    int d = G_INF;
    for (int y = 0; y < ny; ++y) {               // nearest caustic pixel at or below y
        if (caustic_pixel(map, nx, ny, x, y)) d = 0;
        else if (d < G_INF) ++d;
        g[(long long)y * nx + x] = d;
    }
    d = G_INF;
    for (int y = ny - 1; y >= 0; --y) {          // ... or above it
        const int below = g[(long long)y * nx + x];
        if (below == 0) d = 0;
        else if (d < G_INF) ++d;
        if (d < below) g[(long long)y * nx + x] = d;
    }
}

__global__ void __launch_bounds__(BLOCK) k_edt_rows(const int *__restrict__ g, int nx, int ny, double pixel,
                                                    double *__restrict__ out, long long *__restrict__ out_d2)
{
    const long long p = (long long)blockIdx.x * BLOCK + threadIdx.x;
    if (p >= (long long)nx * ny) return;
    const int y = (int)(p / nx), x = (int)(p - (long long)y * nx);
    const int *row = g + (long long)y * nx;
    long long best = (long long)row[x] * row[x];
    const int reach = x > nx - 1 - x ? x : nx - 1 - x;
    for (int dx = 1; dx <= reach; ++dx) {
        const long long dx2 = (long long)dx * dx;
        if (dx2 >= best) break;
        if (x - dx >= 0) {
            const long long gg = row[x - dx];
            const long long c = dx2 + gg * gg;
            if (c < best) best = c;
        }
        if (x + dx < nx) {
            const long long gg = row[x + dx];
            const long long c = dx2 + gg * gg;
            if (c < best) best = c;
        }
    }
    const bool none = best >= (long long)G_INF * G_INF;
    if (out_d2) out_d2[p] = none ? -1 : best;
    out[p] = none ? __longlong_as_double(0x7ff0000000000000ll) : pixel * sqrt((double)best);
}

__global__ void __launch_bounds__(BLOCK) k_directional(const int *__restrict__ map, int nx, int ny, double pixel, int ux,
                                                       int uy, double *__restrict__ out)
{
    const long long p = (long long)blockIdx.x * BLOCK + threadIdx.x;
    if (p >= (long long)nx * ny) return;
    int cy = (int)(p / nx), cx = (int)(p - (long long)cy * nx);
    const int v = map[p];
    const int sx = ux > 0 ? 1 : -1, sy = uy > 0 ? 1 : -1;
    const long long ax = ux > 0 ? ux : -(long long)ux, ay = uy > 0 ? uy : -(long long)uy;
    long long ix = 0, iy = 0;     // borders crossed so far along x and y; the next ones are at (2 i + 1)/|u|
    long long num, den;
    bool hit;
    for (;;) {
        // t_x = (2 ix + 1)/ax against t_y = (2 iy + 1)/ay; a zero component never reaches a border
        const long long lhs = (2 * ix + 1) * ay, rhs = (2 * iy + 1) * ax;
        const bool step_x = ax != 0 && (ay == 0 || lhs <= rhs);
        const bool step_y = ay != 0 && (ax == 0 || rhs <= lhs);
        if (step_x) { num = 2 * ix + 1; den = ax; } else { num = 2 * iy + 1; den = ay; }
        if (step_x) { ++ix; cx += sx; }
        if (step_y) { ++iy; cy += sy; }
        if (cx < 0 || cy < 0 || cx >= nx || cy >= ny) { hit = false; break; }
        if (map[(long long)cy * nx + cx] != v) { hit = true; break; }
    }
    const double ulen = sqrt((double)(ax * ax + ay * ay));
    const double d = pixel * 0.5 * ulen * ((double)num / (double)den);
    out[p] = hit ? d : -d;
}

// Histogram of a distance map by bin and crossing count (the statistics of Fig. 6-7).
// Grid-stride over the pixels, loads coalesced; each CTA counts into its own shared-memory table (when the
// table fits) and adds it to the global one at the end: 64-bit integer atomics, result independent of timing.
constexpr int HIST_SMEM_BINS = 8192;

__global__ void __launch_bounds__(BLOCK) k_distance_histogram(const double *__restrict__ dist, const int *__restrict__ cmap,
                                                              long long P, double bin_width, int num_bins, int num_counts,
                                                              int use_smem, unsigned long long *hist,
                                                              unsigned long long *left_out)
{
    __shared__ unsigned int s_hist[HIST_SMEM_BINS];
    const int table = num_bins * num_counts;
    if (use_smem) {
        for (int i = threadIdx.x; i < table; i += BLOCK) s_hist[i] = 0u;
        __syncthreads();
    }
    unsigned int left = 0;
    for (long long p = (long long)blockIdx.x * BLOCK + threadIdx.x; p < P; p += (long long)gridDim.x * BLOCK) {
        const double d = dist[p];
        if (!(d >= 0.0) || d > 1.79769313486231570e308) { ++left; continue; }
        const double b = floor(__ddiv_rn(d, bin_width));
        if (!(b < (double)num_bins)) { ++left; continue; }
        int row = cmap ? cmap[p] : 0;
        row = row < 0 ? 0 : (row > num_counts - 1 ? num_counts - 1 : row);
        const int at = row * num_bins + (int)b;
        if (use_smem) atomicAdd(&s_hist[at], 1u);
        else atomicAdd(&hist[at], 1ull);
    }
    for (int o = 16; o > 0; o >>= 1) left += __shfl_xor_sync(0xffffffffu, left, o);
    if ((threadIdx.x & 31) == 0 && left) atomicAdd(left_out, (unsigned long long)left);
    if (use_smem) {
        __syncthreads();
        for (int i = threadIdx.x; i < table; i += BLOCK)
            if (s_hist[i]) atomicAdd(&hist[i], (unsigned long long)s_hist[i]);
    }
}

}  // namespace

int distance_histogram_impl(const double *distance, const int32_t *crossing_map, int64_t num_pixels, double bin_width,
                            int32_t num_bins, int32_t num_counts, int64_t *out_hist, int64_t *out_left_out,
                            cudaStream_t stream)
{
    if (!out_hist || !out_left_out || (num_pixels > 0 && !distance)) return invalid("null pointer");
    if (num_pixels < 0 || num_pixels > (1ll << 40)) return invalid("num_pixels out of range");
    if (!(bin_width > 0.0) || !isfinite(bin_width)) return invalid("bin_width");
    if (num_bins < 1 || num_counts < 1 || (long long)num_bins * num_counts > (1ll << 26)) return invalid("table size");
    const long long table = (long long)num_bins * num_counts;
    MLCC_CUDA(cudaMemsetAsync(out_hist, 0, sizeof(int64_t) * table, stream));
    MLCC_CUDA(cudaMemsetAsync(out_left_out, 0, sizeof(int64_t), stream));
    if (num_pixels == 0) return MLCC_OK;
    long long blocks = (num_pixels + BLOCK - 1) / BLOCK;
    const long long cap = 8ll * device_sm_count();        // a CTA counts < 2^32 pixels in its shared table
    if (blocks > cap) blocks = cap;
    k_distance_histogram<<<(unsigned)blocks, BLOCK, 0, stream>>>(distance, crossing_map, (long long)num_pixels, bin_width,
                                                                num_bins, num_counts, table <= HIST_SMEM_BINS ? 1 : 0,
                                                                reinterpret_cast<unsigned long long *>(out_hist),
                                                                reinterpret_cast<unsigned long long *>(out_left_out));
    MLCC_CUDA(cudaGetLastError());
    return MLCC_OK;
}

int distance_map_impl(const int32_t *map, int32_t nx, int32_t ny, double pixel, double *out, int64_t *out_d2,
                      cudaStream_t stream)
{
    if (!map || !out) return invalid("null pointer");
    if (nx < 1 || ny < 1 || (long long)nx * ny > (1ll << 31) || nx > (1 << 24) || ny > (1 << 24))
        return invalid("map size out of range");
    if (!(pixel > 0.0) || !isfinite(pixel)) return invalid("pixel");
    Workspace ws(stream);
    int *g = nullptr;
    cudaError_t e = ws.alloc(&g, (size_t)nx * ny);
    if (e == cudaErrorMemoryAllocation) {
        cudaGetLastError();
        set_last_error("workspace allocation failed");
        return MLCC_ERR_NOMEM;
    }
    MLCC_CUDA(e);
    k_edt_columns<<<(unsigned)((nx + BLOCK - 1) / BLOCK), BLOCK, 0, stream>>>(map, nx, ny, g);
    const long long P = (long long)nx * ny;
    k_edt_rows<<<(unsigned)((P + BLOCK - 1) / BLOCK), BLOCK, 0, stream>>>(g, nx, ny, pixel, out,
                                                                          reinterpret_cast<long long *>(out_d2));
    MLCC_CUDA(cudaGetLastError());
    return MLCC_OK;
}

int directional_distance_map_impl(const int32_t *map, int32_t nx, int32_t ny, double pixel, int32_t ux, int32_t uy,
                                  double *out, cudaStream_t stream)
{
    if (!map || !out) return invalid("null pointer");
    if (nx < 1 || ny < 1 || (long long)nx * ny > (1ll << 31) || nx > (1 << 24) || ny > (1 << 24))
        return invalid("map size out of range");
    if (!(pixel > 0.0) || !isfinite(pixel)) return invalid("pixel");
    if (ux == 0 && uy == 0) return invalid("direction (0, 0)");
    if (ux > (1 << 20) || ux < -(1 << 20) || uy > (1 << 20) || uy < -(1 << 20)) return invalid("direction component > 2^20");
    const long long P = (long long)nx * ny;
    k_directional<<<(unsigned)((P + BLOCK - 1) / BLOCK), BLOCK, 0, stream>>>(map, nx, ny, pixel, ux, uy, out);
    MLCC_CUDA(cudaGetLastError());
    return MLCC_OK;
}

}  // namespace mlcc
