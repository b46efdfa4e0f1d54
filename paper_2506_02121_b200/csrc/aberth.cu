// aberth.cu — critical curves by batched, masked Aberth–Ehrlich iterations with phase continuation.
//
// What it computes (Eq. 15 with alpha_s = -kappa_star z):
//   F(z,phi) = gamma + S2 - (1-kappa_s) e^{-i phi},  S2 = sum_i m_i/(z-z_i)^2,
//   F'(z)    = -2 S3,                                S3 = sum_i m_i/(z-z_i)^3,
//   P'/P     = F'/F + 2 S1 (Eq. 19),   S1 = sum_i 1/(z-z_i),
//   Aberth–Ehrlich (Eq. 17), multiplied through by F:
//   Delta_k  = F / (F' + F (2 S1 - A)),  A = sum_{r != k} 1/(z_k - z_r),  z_k <- z_k - Delta_k,
//   root k frozen once |Delta_k| < tol.
//
// Organisation:
//   * The rows [0, num_phi) are cut into sub-chains; each sub-chain cold-starts its centre row from
//     z_i +/- 1 and then grows towards both ends.  One "step"
//     advances every growing direction ("slot") by one row; all slots of a step are iterated
//     together by the same kernels, so the grid is full even when 2N is small.
//   * A device-side state machine (DevState) decides what each launch does; the host only enqueues
//     [seed, compute, apply, finalize] groups and polls one flag per chunk.  No host round trip
//     sits inside the iteration loop.
//   * compute: one CTA per tile of unfrozen roots of one slot.  Each root's sums are split over
//     T threads (T = 1..256, chosen on the device from the number of unfrozen roots so that the
//     machine stays full when few roots are left); stars and the slot's current roots stream
//     through shared memory.  Jacobi: updates go to a separate buffer and are applied by `apply`,
//     which also compacts the list of unfrozen roots.
#include "mlcc_common.cuh"

#include <math.h>
#include <vector>

namespace mlcc {
namespace {

constexpr int BLOCK = 256;        // threads per CTA of the compute kernel
constexpr int TILE = 1024;        // sources staged in shared memory per tile
constexpr int MAX_ORDER = 5;      // highest predictor order
constexpr int MAX_SLOTS = 1024;   // most slots in one step (2 per sub-chain)
constexpr double TINY = 1e-300;   // added to |d|^2: makes the self pair finite, invisible otherwise
#ifndef MLCC_U_STAR
#define MLCC_U_STAR 4
#endif
#ifndef MLCC_U_ROOT
#define MLCC_U_ROOT 8
#endif
#ifndef MLCC_MIN_BLOCKS
#define MLCC_MIN_BLOCKS 2
#endif
constexpr int U_STAR = MLCC_U_STAR;   // pairs in flight per thread in the star loop
constexpr int U_ROOT = MLCC_U_ROOT;   // ... in the root loop (even)

struct DevState {
    int step;             // current step: 0 = cold centre rows, s >= 1 = rows centre +/- s
    int iter;             // iterations done in this step
    int n_slots;          // slots active in this step
    int done;             // all steps finished
    int need_seed;        // the seed kernel must write starting values for this step
    int cur;              // which of the two active lists is current
    int T;                // threads per root of the next compute launch
    int n_tiles;          // CTA tiles of the next compute launch
    int total_active;     // unfrozen roots over all slots
    int total_iterations;
    int unconverged_rows;
    int degenerate;
    long long root_iterations;
    long long launches_used;  // compute launches that did work
};

struct Params {
    // problem
    const double2 *stars;     // [N]
    const double *masses;     // [N]
    int N;
    int n_r;                  // 2N
    double gamma;
    double tol2;              // tol^2
    int max_iter;
    int max_iter_cold;
    int order;                // predictor order
    int min_T;
    int target_threads;       // threads the compute grid can keep resident
    const double2 *rot;       // [num_phi]  (1-kappa_s) e^{-i phi_j}
    const double2 *init_roots;  // [n_r] or null
    double2 *roots;           // [num_phi][n_r]
    int *out_iters;           // [num_phi] or null
    int *out_unconverged;     // [num_phi] or null
    // plan
    int n_sub;                // sub-chains
    const long long *sub_first;   // [n_sub]
    const long long *sub_centre;  // [n_sub]
    const long long *sub_end;     // [n_sub]
    int max_steps;            // largest distance from a centre to an end of its sub-chain
    // workspace
    DevState *state;
    long long *slot_row;      // [MAX_SLOTS] row solved by the slot in this step
    int *slot_sub;            // [MAX_SLOTS] sub-chain of the slot
    int *slot_dir;            // [MAX_SLOTS] -1, +1 (0 = centre)
    int *slot_iters;          // [MAX_SLOTS] iteration at which the slot last had unfrozen roots
    int *n_active;            // [2][MAX_SLOTS]
    int *tile_start;          // [MAX_SLOTS + 1]
    int *list;                // [2][max_slots][n_r]
    double2 *delta;           // [max_slots][n_r]
    int max_slots;            // slots that can be live at once (2 n_sub)
};

// ------------------------------------------------------------------------------------------------
// pair bodies
// ------------------------------------------------------------------------------------------------

// (root, star): accumulates S1 += 1/d, S2 += m/d^2, S3 += m/d^3 with d = z - z_i.
// w = 1/d = conj(d)/|d|^2; dy is taken as (y_i - y) so that w = (dx, dy) * inv.
__device__ __forceinline__ void pair_star(double zx, double zy, double2 s, double m,
                                          double &s1x, double &s1y, double &s2x, double &s2y,
                                          double &s3x, double &s3y)
{
    double dx = zx - s.x;
    double dy = s.y - zy;
    double r2 = fma(dy, dy, fma(dx, dx, TINY));
    double inv = rcp_full(r2);
    double wx = dx * inv;
    double wy = dy * inv;
    s1x += wx;
    s1y += wy;
    double ux = m * wx;
    double uy = m * wy;
    double qx = fma(-uy, wy, ux * wx);   // q = m w^2
    double qy = fma(ux, wy, uy * wx);
    s2x += qx;
    s2y += qy;
    s3x = fma(qx, wx, s3x);               // S3 += q w
    s3x = fma(-qy, wy, s3x);
    s3y = fma(qx, wy, s3y);
    s3y = fma(qy, wx, s3y);
}

// (root, root): A += 1/(z_k - z_r).  Only the convergence RATE depends on A (the fixed point of
// the update is F = 0 whatever A is), so the 20-bit reciprocal seed is used as it is.  A root
// paired with itself has d = 0 exactly: |d|^2 + TINY = 1e-300, the seed is finite, and the pair
// contributes conj(d) * inv = 0.  For every other pair TINY is lost in the rounding of |d|^2.
__device__ __forceinline__ void pair_root(double zx, double zy, double2 r, double &ax, double &ay)
{
    double dx = zx - r.x;
    double dy = r.y - zy;
    double r2 = fma(dy, dy, fma(dx, dx, TINY));
    double inv = rcp_seed(r2);
    ax = fma(dx, inv, ax);
    ay = fma(dy, inv, ay);
}

// ------------------------------------------------------------------------------------------------
// seed kernel: starting values of every slot's new row + identity active lists
// ------------------------------------------------------------------------------------------------
__constant__ double c_coef[MAX_ORDER + 1][MAX_ORDER + 1] = {
    {1, 0, 0, 0, 0, 0},          {2, -1, 0, 0, 0, 0},          {3, -3, 1, 0, 0, 0},
    {4, -6, 4, -1, 0, 0},        {5, -10, 10, -5, 1, 0},       {6, -15, 20, -15, 6, -1}};

__global__ void k_seed(Params p)
{
    const DevState st = *p.state;
    if (st.done || !st.need_seed) return;
    const long long total = (long long)st.n_slots * p.n_r;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int slot = (int)(idx / p.n_r);
        const int k = (int)(idx - (long long)slot * p.n_r);
        const long long row = p.slot_row[slot];
        double2 z;
        if (st.step == 0) {
            if (p.init_roots) {
                z = p.init_roots[k];
            } else {  // z_i + 1, z_i - 1
                const int i = (k < p.N) ? k : k - p.N;
                z = p.stars[i];
                z.x += (k < p.N) ? 1.0 : -1.0;
            }
        } else {
            // extrapolate through the last (order+1) rows of this chain that exist:
            // rows row - dir*q, q = 1 .. avail, lie inside the sub-chain and were solved in earlier steps
            const int sub = p.slot_sub[slot];
            const int dir = p.slot_dir[slot];
            long long room = (dir > 0) ? (row - p.sub_first[sub]) : (p.sub_end[sub] - 1 - row);
            long long avail = min((long long)(2 * st.step - 1), room);
            int order = (int)min((long long)p.order, avail - 1);
            double zx = 0.0, zy = 0.0;
            for (int q = order; q >= 0; --q) {
                const double2 v = p.roots[(row - (long long)dir * (q + 1)) * p.n_r + k];
                zx = fma(c_coef[order][q], v.x, zx);
                zy = fma(c_coef[order][q], v.y, zy);
            }
            z = make_double2(zx, zy);
        }
        p.roots[row * p.n_r + k] = z;
        p.list[((long long)st.cur * p.max_slots + slot) * p.n_r + k] = k;
    }
}

// ------------------------------------------------------------------------------------------------
// compute kernel
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(BLOCK, MLCC_MIN_BLOCKS) k_compute(Params p)
{
    __shared__ double2 s_xy[TILE];
    __shared__ double s_m[TILE];
    __shared__ double s_red[BLOCK / 32][6];

    const DevState st = *p.state;
    if (st.done) return;
    const int T = st.T;                 // threads per root (power of two, 1..256)
    const int TL = T < 32 ? T : 32;     // of which inside one warp
    const int W = T / TL;               // warps per root
    const int roots_per_tile = BLOCK / T;
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    // position of this thread's root inside the tile, and which share of the sources it sums
    const int local_root = (warp / W) * (32 / TL) + lane / TL;
    const int sub = (warp % W) * TL + (lane % TL);
    const int* n_active = p.n_active + st.cur * MAX_SLOTS;

    for (int tile = blockIdx.x; tile < st.n_tiles; tile += gridDim.x) {
        // slot of this tile: last slot with tile_start <= tile
        int lo = 0, hi = st.n_slots;
        while (hi - lo > 1) {
            int mid = (lo + hi) >> 1;
            if (p.tile_start[mid] <= tile) lo = mid; else hi = mid;
        }
        const int slot = lo;
        const long long row = p.slot_row[slot];
        const double2 *zrow = p.roots + row * p.n_r;
        const int *list = p.list + ((long long)st.cur * p.max_slots + slot) * p.n_r;
        const int pos = (tile - p.tile_start[slot]) * roots_per_tile + local_root;
        const bool valid = pos < n_active[slot];
        int k = 0;
        double zx = 0.0, zy = 0.0;
        if (valid) {
            k = list[pos];
            const double2 z = zrow[k];
            zx = z.x;
            zy = z.y;
        }
        double s1x = 0, s1y = 0, s2x = 0, s2y = 0, s3x = 0, s3y = 0, ax = 0, ay = 0, bx = 0, by = 0;

        // ---- stars ----
        for (int base = 0; base < p.N; base += TILE) {
            const int cnt = min(TILE, p.N - base);
            __syncthreads();
            for (int i = tid; i < cnt; i += BLOCK) {
                s_xy[i] = p.stars[base + i];
                s_m[i] = p.masses[base + i];
            }
            __syncthreads();
            if (valid) {
                // blocks of U_STAR independent pairs with no exit in between, so that their
                // dependent chains (|d|^2 -> reciprocal -> powers) interleave; then the ragged tail
                int j = sub;
                for (; j + (U_STAR - 1) * T < cnt; j += U_STAR * T) {
                    double2 s[U_STAR];
                    double m[U_STAR];
#pragma unroll
                    for (int u = 0; u < U_STAR; ++u) { s[u] = s_xy[j + u * T]; m[u] = s_m[j + u * T]; }
#pragma unroll
                    for (int u = 0; u < U_STAR; ++u)
                        pair_star(zx, zy, s[u], m[u], s1x, s1y, s2x, s2y, s3x, s3y);
                }
                for (; j < cnt; j += T)
                    pair_star(zx, zy, s_xy[j], s_m[j], s1x, s1y, s2x, s2y, s3x, s3y);
            }
        }
        // ---- the other roots of this row (frozen ones included) ----
        for (int base = 0; base < p.n_r; base += TILE) {
            const int cnt = min(TILE, p.n_r - base);
            __syncthreads();
            for (int i = tid; i < cnt; i += BLOCK) s_xy[i] = zrow[base + i];
            __syncthreads();
            if (valid) {
                int j = sub;
                for (; j + (U_ROOT - 1) * T < cnt; j += U_ROOT * T) {
                    double2 r[U_ROOT];
#pragma unroll
                    for (int u = 0; u < U_ROOT; ++u) r[u] = s_xy[j + u * T];
#pragma unroll
                    for (int u = 0; u < U_ROOT; u += 2) {   // two accumulator chains
                        pair_root(zx, zy, r[u], ax, ay);
                        pair_root(zx, zy, r[u + 1], bx, by);
                    }
                }
                for (; j < cnt; j += T) pair_root(zx, zy, s_xy[j], ax, ay);
            }
        }
        // ---- reduce the T partial sums ----
        double tx = 2.0 * s1x - (ax + bx);   // 2 S1 - A
        double ty = 2.0 * s1y - (ay + by);
        for (int o = TL >> 1; o > 0; o >>= 1) {
            s2x += __shfl_xor_sync(0xffffffffu, s2x, o);
            s2y += __shfl_xor_sync(0xffffffffu, s2y, o);
            s3x += __shfl_xor_sync(0xffffffffu, s3x, o);
            s3y += __shfl_xor_sync(0xffffffffu, s3y, o);
            tx += __shfl_xor_sync(0xffffffffu, tx, o);
            ty += __shfl_xor_sync(0xffffffffu, ty, o);
        }
        if (W > 1) {
            __syncthreads();
            if (lane == 0) {
                s_red[warp][0] = s2x; s_red[warp][1] = s2y; s_red[warp][2] = s3x;
                s_red[warp][3] = s3y; s_red[warp][4] = tx;  s_red[warp][5] = ty;
            }
            __syncthreads();
            if (warp % W == 0 && lane == 0) {
                for (int w2 = 1; w2 < W; ++w2) {
                    s2x += s_red[warp + w2][0]; s2y += s_red[warp + w2][1];
                    s3x += s_red[warp + w2][2]; s3y += s_red[warp + w2][3];
                    tx += s_red[warp + w2][4];  ty += s_red[warp + w2][5];
                }
            }
        }
        // ---- Aberth step ----
        if (valid && sub == 0) {
            const double2 rot = p.rot[row];
            const double fx = p.gamma + s2x - rot.x;   // F
            const double fy = s2y - rot.y;
            const double gx = -2.0 * s3x;               // F'
            const double gy = -2.0 * s3y;
            const double dnx = gx + (fx * tx - fy * ty);  // F' + F (2 S1 - A)
            const double dny = gy + (fx * ty + fy * tx);
            const double dn2 = dnx * dnx + dny * dny;
            double2 d;
            d.x = (fx * dnx + fy * dny) / dn2;          // F / den
            d.y = (fy * dnx - fx * dny) / dn2;
            p.delta[(long long)slot * p.n_r + pos] = d;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// apply kernel: z_k -= Delta_k, freeze converged roots, compact the list of unfrozen roots
// grid: (ceil(n_r / BLOCK), max_slots)
// ------------------------------------------------------------------------------------------------
__global__ void k_apply(Params p)
{
    const DevState st = *p.state;
    if (st.done) return;
    const int slot = blockIdx.y;
    if (slot >= st.n_slots) return;
    const int n_act = p.n_active[st.cur * MAX_SLOTS + slot];
    const int pos = blockIdx.x * blockDim.x + threadIdx.x;
    if (blockIdx.x * blockDim.x >= n_act) return;
    const int *list = p.list + ((long long)st.cur * p.max_slots + slot) * p.n_r;
    int *next = p.list + ((long long)(st.cur ^ 1) * p.max_slots + slot) * p.n_r;
    bool keep = false;
    int k = 0;
    if (pos < n_act) {
        k = list[pos];
        const double2 d = p.delta[(long long)slot * p.n_r + pos];
        const double d2 = d.x * d.x + d.y * d.y;
        double2 *zp = p.roots + p.slot_row[slot] * p.n_r + k;
        if (d2 <= 1.79769313486231570e308) {   // finite step
            double2 z = *zp;
            z.x -= d.x;
            z.y -= d.y;
            *zp = z;
            keep = !(d2 < p.tol2);
        } else {                                // NaN / Inf: freeze where it is, report
            atomicAdd(&p.state->degenerate, 1);
        }
    }
    const unsigned mask = __ballot_sync(0xffffffffu, keep);
    const int lane = threadIdx.x & 31;
    int base = 0;
    if (lane == 0 && mask) base = atomicAdd(&p.n_active[(st.cur ^ 1) * MAX_SLOTS + slot], __popc(mask));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (keep) next[base + __popc(mask & ((1u << lane) - 1u))] = k;
}

// ------------------------------------------------------------------------------------------------
// finalize kernel (one block): advances the state machine
// ------------------------------------------------------------------------------------------------
__device__ int pick_T(const Params &p, int total_active)
{
    int T = 1;
    while (T < 256 && (long long)total_active * T * 2 <= p.target_threads) T <<= 1;
    if (T < p.min_T) T = p.min_T;
    return T;
}

// one thread: tile table for the counts in n_active[cur]
__device__ void build_tiles(const Params &p, DevState &st)
{
    const int *n_active = p.n_active + st.cur * MAX_SLOTS;
    int total = 0;
    for (int s = 0; s < st.n_slots; ++s) total += n_active[s];
    st.total_active = total;
    st.T = pick_T(p, total);
    const int rpt = BLOCK / st.T;
    int t = 0;
    for (int s = 0; s < st.n_slots; ++s) {
        p.tile_start[s] = t;
        t += (n_active[s] + rpt - 1) / rpt;
    }
    p.tile_start[st.n_slots] = t;
    st.n_tiles = t;
}

// one thread: slots of step st.step
__device__ void build_slots(const Params &p, DevState &st)
{
    int n = 0;
    if (st.step == 0) {
        for (int c = 0; c < p.n_sub; ++c) {
            p.slot_row[n] = p.sub_centre[c];
            p.slot_sub[n] = c;
            p.slot_dir[n] = 0;
            ++n;
        }
    } else {
        for (int c = 0; c < p.n_sub; ++c) {
            const long long up = p.sub_centre[c] + st.step, dn = p.sub_centre[c] - st.step;
            if (dn >= p.sub_first[c]) { p.slot_row[n] = dn; p.slot_sub[n] = c; p.slot_dir[n] = -1; ++n; }
            if (up < p.sub_end[c])    { p.slot_row[n] = up; p.slot_sub[n] = c; p.slot_dir[n] = +1; ++n; }
        }
    }
    st.n_slots = n;
    for (int s = 0; s < n; ++s) {
        p.n_active[st.cur * MAX_SLOTS + s] = p.n_r;
        p.n_active[(st.cur ^ 1) * MAX_SLOTS + s] = 0;
        p.slot_iters[s] = 0;
    }
    st.iter = 0;
    st.need_seed = 1;
    if (n == 0) st.done = 1;
}

// input check: flags[0] = non-finite star coordinates / masses, flags[1] = pairs of coincident stars
// (two stars at the same point make P(z) lose two roots: the degree claim 2N fails)
__global__ void k_check_stars(const double2 *__restrict__ stars, const double *__restrict__ masses, int N,
                              int *flags)
{
    __shared__ double2 s_xy[BLOCK];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double2 me = make_double2(0.0, 0.0);
    if (i < N) {
        me = stars[i];
        const double m = masses[i];
        if (!(fabs(me.x) <= 1e300) || !(fabs(me.y) <= 1e300) || !(fabs(m) <= 1e300)) atomicAdd(&flags[0], 1);
    }
    int same = 0;
    for (int base = 0; base < N; base += BLOCK) {
        __syncthreads();
        if (base + threadIdx.x < N) s_xy[threadIdx.x] = stars[base + threadIdx.x];
        __syncthreads();
        const int cnt = min(BLOCK, N - base);
        if (i < N)
            for (int j = 0; j < cnt; ++j)
                if (base + j < i && s_xy[j].x == me.x && s_xy[j].y == me.y) ++same;
    }
    if (same) atomicAdd(&flags[1], same);
}

__global__ void k_init(Params p)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    DevState st;
    st.step = 0; st.iter = 0; st.n_slots = 0; st.done = 0; st.need_seed = 1; st.cur = 0;
    st.T = 1; st.n_tiles = 0; st.total_active = 0; st.total_iterations = 0;
    st.unconverged_rows = 0; st.degenerate = 0; st.root_iterations = 0; st.launches_used = 0;
    build_slots(p, st);
    build_tiles(p, st);
    *p.state = st;
}

__global__ void k_finalize(Params p)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    DevState st = *p.state;
    if (st.done) return;
    // the iteration that just ran
    st.iter += 1;
    st.total_iterations += 1;
    st.root_iterations += st.total_active;
    st.launches_used += 1;
    st.need_seed = 0;
    int *cur = p.n_active + st.cur * MAX_SLOTS;
    int *nxt = p.n_active + (st.cur ^ 1) * MAX_SLOTS;
    int remaining = 0;
    for (int s = 0; s < st.n_slots; ++s) {
        if (cur[s] > 0) p.slot_iters[s] = st.iter;
        remaining += nxt[s];
        cur[s] = 0;   // becomes the "next" counter of the following iteration
    }
    st.cur ^= 1;
    const int cap = (st.step == 0) ? p.max_iter_cold : p.max_iter;
    if (remaining == 0 || st.iter >= cap) {
        // step finished: per-row diagnostics, then the next step's slots
        for (int s = 0; s < st.n_slots; ++s) {
            const long long row = p.slot_row[s];
            const int left = p.n_active[st.cur * MAX_SLOTS + s];
            if (p.out_iters) p.out_iters[row] = p.slot_iters[s];
            if (p.out_unconverged) p.out_unconverged[row] = left;
            if (left > 0) st.unconverged_rows += 1;
        }
        st.step += 1;
        if (st.step > p.max_steps) { st.done = 1; st.n_slots = 0; }
        else build_slots(p, st);
    }
    if (!st.done) build_tiles(p, st);
    *p.state = st;
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
int plan_subchains_host(int64_t N, int64_t num_phi, int32_t num_subchains, int32_t capacity,
                        int64_t *first_row, int64_t *centre_row, int64_t *end_row)
{
    if (N < 1 || num_phi < 1 || num_subchains < 0) return -MLCC_ERR_INVALID_ARG;
    int64_t n = num_subchains;
    if (n == 0) {
        // enough slots (2 per sub-chain) to keep ~3e5 roots in flight, but chains at least 16 rows long
        const int64_t n_r = 2 * N;
        int64_t slots = (300000 + n_r - 1) / n_r;
        n = (slots + 1) / 2;
        const int64_t by_len = num_phi / 16;
        if (n > by_len) n = by_len;
    }
    if (n > num_phi) n = num_phi;
    if (n > MAX_SLOTS / 2) n = MAX_SLOTS / 2;
    if (n < 1) n = 1;
    if (capacity < n) return -MLCC_ERR_INVALID_ARG;
    for (int64_t c = 0; c < n; ++c) {
        const int64_t a = (num_phi * c) / n, b = (num_phi * (c + 1)) / n;
        first_row[c] = a;
        end_row[c] = b;
        centre_row[c] = a + (b - a) / 2;
    }
    return (int)n;
}

int critical_curves_impl(const double *star_xy, const double *masses, int64_t N, double kappa_s,
                         double gamma, int64_t num_phi, double tol, int32_t max_iter,
                         double *out_roots, const mlcc_options *opt_in, const double *init_roots,
                         int32_t *out_iters, int32_t *out_unconverged, mlcc_stats *out_stats,
                         cudaStream_t stream)
{
    if (!star_xy || !masses || !out_roots) return invalid("null pointer");
    if (N < 1 || N > (1 << 29)) return invalid("N out of range");
    if (num_phi < 1) return invalid("num_phi < 1");
    if (!(tol > 0.0) || !isfinite(tol)) return invalid("tol must be positive and finite");
    if (max_iter < 1) return invalid("max_iter < 1");
    if (!isfinite(kappa_s) || !isfinite(gamma)) return invalid("kappa_s / gamma not finite");
    mlcc_options opt;
    mlcc_options_default(&opt);
    if (opt_in) {
        if (opt_in->struct_size != 0 && opt_in->struct_size != (int32_t)sizeof(mlcc_options))
            return invalid("mlcc_options.struct_size");
        opt = *opt_in;
    }
    const int64_t phi_total = opt.phi_index_total > 0 ? opt.phi_index_total : num_phi;
    const int64_t phi_off = opt.phi_index_offset;
    int order = opt.predictor_order < 0 ? 3 : opt.predictor_order;
    if (order > MAX_ORDER) return invalid("predictor_order > 5");
    int min_T = opt.min_lanes_per_root <= 0 ? 1 : opt.min_lanes_per_root;
    if (min_T > 256 || (min_T & (min_T - 1))) return invalid("min_lanes_per_root must be a power of two <= 256");
    if (opt.num_subchains < 0 || opt.max_iter_cold < 0) return invalid("negative option");

    // phase table (1-kappa_s) e^{-i phi_j}; c(phi_j) = 0 on a row is rejected (degree drop)
    std::vector<double2> rot((size_t)num_phi);
    const double two_pi = 6.283185307179586476925286766559;
    for (int64_t j = 0; j < num_phi; ++j) {
        const double phi = two_pi * (double)(j + phi_off) / (double)phi_total;
        rot[(size_t)j].x = (1.0 - kappa_s) * cos(phi);
        rot[(size_t)j].y = -(1.0 - kappa_s) * sin(phi);
        const double cx = rot[(size_t)j].x - gamma, cy = rot[(size_t)j].y;
        if (cx == 0.0 && cy == 0.0) return invalid("c(phi_j) = (1-kappa_s) e^{-i phi_j} - gamma vanishes on a grid row");
    }
    if (1.0 - kappa_s == 0.0 && gamma == 0.0) return invalid("kappa_s = 1 and gamma = 0");

    // plan
    std::vector<long long> first(MAX_SLOTS), centre(MAX_SLOTS), end(MAX_SLOTS);
    std::vector<int64_t> f64v(MAX_SLOTS), c64v(MAX_SLOTS), e64v(MAX_SLOTS);
    const int n_sub = plan_subchains_host(N, num_phi, opt.num_subchains, MAX_SLOTS / 2, f64v.data(),
                                          c64v.data(), e64v.data());
    if (n_sub < 1) return invalid("num_subchains");
    int max_steps = 0;
    for (int c = 0; c < n_sub; ++c) {
        first[c] = f64v[c]; centre[c] = c64v[c]; end[c] = e64v[c];
        const long long a = centre[c] - first[c], b = end[c] - 1 - centre[c];
        if (a > max_steps) max_steps = (int)a;
        if (b > max_steps) max_steps = (int)b;
    }
    const int max_slots = 2 * n_sub > 1 ? 2 * n_sub : 1;
    const int n_r = (int)(2 * N);

    Workspace ws(stream);
    Params p{};
    double2 *d_rot = nullptr;
    long long *d_plan = nullptr;
    cudaError_t e;
    if ((e = ws.alloc(&d_rot, (size_t)num_phi)) != cudaSuccess ||
        (e = ws.alloc(&d_plan, (size_t)3 * n_sub)) != cudaSuccess ||
        (e = ws.alloc(&p.state, 1)) != cudaSuccess ||
        (e = ws.alloc(&p.slot_row, MAX_SLOTS)) != cudaSuccess ||
        (e = ws.alloc(&p.slot_sub, MAX_SLOTS)) != cudaSuccess ||
        (e = ws.alloc(&p.slot_dir, MAX_SLOTS)) != cudaSuccess ||
        (e = ws.alloc(&p.slot_iters, MAX_SLOTS)) != cudaSuccess ||
        (e = ws.alloc(&p.n_active, 2 * MAX_SLOTS)) != cudaSuccess ||
        (e = ws.alloc(&p.tile_start, MAX_SLOTS + 1)) != cudaSuccess ||
        (e = ws.alloc(&p.list, (size_t)2 * max_slots * n_r)) != cudaSuccess ||
        (e = ws.alloc(&p.delta, (size_t)max_slots * n_r)) != cudaSuccess) {
        if (e == cudaErrorMemoryAllocation) {
            cudaGetLastError();
            set_last_error("workspace allocation failed");
            return MLCC_ERR_NOMEM;
        }
        return cuda_fail(e, "cudaMallocAsync", __FILE__, __LINE__);
    }
    MLCC_CUDA(cudaMemcpyAsync(d_rot, rot.data(), sizeof(double2) * (size_t)num_phi,
                              cudaMemcpyHostToDevice, stream));
    std::vector<long long> plan((size_t)3 * n_sub);
    for (int c = 0; c < n_sub; ++c) { plan[c] = first[c]; plan[n_sub + c] = centre[c]; plan[2 * n_sub + c] = end[c]; }
    MLCC_CUDA(cudaMemcpyAsync(d_plan, plan.data(), sizeof(long long) * plan.size(),
                              cudaMemcpyHostToDevice, stream));
    MLCC_CUDA(cudaMemsetAsync(p.n_active, 0, sizeof(int) * 2 * MAX_SLOTS, stream));

    // input check (one small read-back before the solve)
    {
        int *d_flags = nullptr;
        MLCC_CUDA(ws.alloc(&d_flags, 2));
        MLCC_CUDA(cudaMemsetAsync(d_flags, 0, 2 * sizeof(int), stream));
        k_check_stars<<<(unsigned)((N + BLOCK - 1) / BLOCK), BLOCK, 0, stream>>>(
            reinterpret_cast<const double2 *>(star_xy), masses, (int)N, d_flags);
        int h_flags[2] = {0, 0};
        MLCC_CUDA(cudaMemcpyAsync(h_flags, d_flags, 2 * sizeof(int), cudaMemcpyDeviceToHost, stream));
        MLCC_CUDA(cudaStreamSynchronize(stream));
        MLCC_CUDA(cudaGetLastError());
        if (h_flags[0]) return invalid("non-finite star position or mass");
        if (h_flags[1]) {
            set_last_error("coincident stars: P(z) loses roots (merge them into one star of the summed mass)");
            return MLCC_ERR_DEGENERATE;
        }
    }

    int blocks_per_sm = 0;
    MLCC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, k_compute, BLOCK, 0));
    if (blocks_per_sm < 1) blocks_per_sm = 1;
    const int sms = device_sm_count();
    const int grid_compute = sms * blocks_per_sm;

    p.stars = reinterpret_cast<const double2 *>(star_xy);
    p.masses = masses;
    p.N = (int)N;
    p.n_r = n_r;
    p.gamma = gamma;
    p.tol2 = tol * tol;
    p.max_iter = max_iter;
    p.max_iter_cold = opt.max_iter_cold > 0 ? opt.max_iter_cold : max_iter;
    p.order = order;
    p.min_T = min_T;
    p.target_threads = grid_compute * BLOCK;
    p.rot = d_rot;
    p.init_roots = reinterpret_cast<const double2 *>(init_roots);
    p.roots = reinterpret_cast<double2 *>(out_roots);
    p.out_iters = out_iters;
    p.out_unconverged = out_unconverged;
    p.n_sub = n_sub;
    p.sub_first = d_plan;
    p.sub_centre = d_plan + n_sub;
    p.sub_end = d_plan + 2 * n_sub;
    p.max_steps = max_steps;
    p.max_slots = max_slots;

    cudaEvent_t ev0 = nullptr, ev1 = nullptr, ev_poll[2] = {nullptr, nullptr};
    MLCC_CUDA(cudaEventCreate(&ev0));
    MLCC_CUDA(cudaEventCreate(&ev1));
    MLCC_CUDA(cudaEventCreateWithFlags(&ev_poll[0], cudaEventDisableTiming));
    MLCC_CUDA(cudaEventCreateWithFlags(&ev_poll[1], cudaEventDisableTiming));
    DevState *h_state = nullptr;   // pinned, two snapshots
    MLCC_CUDA(cudaMallocHost(&h_state, 2 * sizeof(DevState)));
    h_state[0].done = h_state[1].done = 0;

    MLCC_CUDA(cudaEventRecord(ev0, stream));
    k_init<<<1, 32, 0, stream>>>(p);
    const int grid_seed = sms * 4;
    const dim3 grid_apply((unsigned)((n_r + BLOCK - 1) / BLOCK), (unsigned)max_slots);
    int64_t launches = 1;
    // Upper bound on iteration groups, so that a device-side fault cannot spin the host forever.
    const long long max_groups = (long long)(max_steps + 1) * (long long)(p.max_iter > p.max_iter_cold ? p.max_iter : p.max_iter_cold) + 8;
    const int chunk = 16;
    long long groups = 0;
    int which = 0;
    bool finished = false;
    int rc = MLCC_OK;
    while (!finished && groups < max_groups + 2 * chunk) {
        for (int g = 0; g < chunk; ++g) {
            k_seed<<<grid_seed, BLOCK, 0, stream>>>(p);
            k_compute<<<grid_compute, BLOCK, 0, stream>>>(p);
            k_apply<<<grid_apply, BLOCK, 0, stream>>>(p);
            k_finalize<<<1, 32, 0, stream>>>(p);
        }
        launches += 4 * chunk;
        groups += chunk;
        cudaMemcpyAsync(&h_state[which], p.state, sizeof(DevState), cudaMemcpyDeviceToHost, stream);
        cudaEventRecord(ev_poll[which], stream);
        // look at the previous chunk's snapshot while this one runs
        if (groups > chunk) {
            cudaError_t es = cudaEventSynchronize(ev_poll[which ^ 1]);
            if (es != cudaSuccess) { rc = cuda_fail(es, "cudaEventSynchronize", __FILE__, __LINE__); break; }
            if (h_state[which ^ 1].done) finished = true;
        }
        which ^= 1;
    }
    DevState fin{};
    if (rc == MLCC_OK) {
        cudaEventRecord(ev1, stream);
        cudaError_t es = cudaMemcpyAsync(&h_state[0], p.state, sizeof(DevState), cudaMemcpyDeviceToHost, stream);
        if (es == cudaSuccess) es = cudaStreamSynchronize(stream);
        if (es == cudaSuccess) es = cudaGetLastError();
        if (es != cudaSuccess) rc = cuda_fail(es, "critical-curve kernels", __FILE__, __LINE__);
        else fin = h_state[0];
    }
    float ms = 0.f;
    if (rc == MLCC_OK) cudaEventElapsedTime(&ms, ev0, ev1);
    cudaEventDestroy(ev0); cudaEventDestroy(ev1);
    cudaEventDestroy(ev_poll[0]); cudaEventDestroy(ev_poll[1]);
    cudaFreeHost(h_state);
    if (rc != MLCC_OK) return rc;
    if (!fin.done) {
        set_last_error("internal: state machine did not finish");
        return MLCC_ERR_CUDA;
    }
    if (out_stats) {
        out_stats->root_iterations = fin.root_iterations;
        out_stats->star_pairs = fin.root_iterations * N;
        out_stats->root_pairs = fin.root_iterations * (2 * N - 1);
        out_stats->kernel_launches = launches;
        out_stats->total_iterations = fin.total_iterations;
        out_stats->steps = max_steps + 1;
        out_stats->subchains = n_sub;
        out_stats->predictor_order = order;
        out_stats->unconverged_rows = fin.unconverged_rows;
        out_stats->degenerate_roots = fin.degenerate;
        out_stats->solve_ms = ms;
        out_stats->reserved = 0.f;
    }
    if (fin.degenerate > 0) {
        set_last_error("NaN/Inf Aberth step: a root landed on a star or another root, or stars coincide");
        return MLCC_ERR_DEGENERATE;
    }
    if (fin.unconverged_rows > 0) {
        set_last_error("some roots were still unfrozen at max_iter");
        return MLCC_ERR_NOT_CONVERGED;
    }
    return MLCC_OK;
}

}  // namespace mlcc
