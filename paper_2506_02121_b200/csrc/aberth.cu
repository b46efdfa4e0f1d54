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
// Organisation (DESIGN.md "Driver" and "Kernels"):
//   * The rows [0, num_phi) are cut into sub-chains; each sub-chain cold-starts its centre row from
//     z_i +/- 1 and then grows towards both ends.  One "step"
//     starts one new row in every growing direction; a row being solved occupies a "slot", and all
//     live slots are iterated together by the same kernels, so the grid is full even when 2N is small.
//     Steps are pipelined: the next one starts as soon as the newest has (almost) only nearly
//     converged roots left, and the stragglers of older rows ride along as extra slots.
//   * A device-side state machine (DevState, finalize_iteration) decides what each launch does; the
//     host only enqueues [seed, compute, compute without A, apply count, apply write] groups and polls
//     one flag per chunk.  No host round trip sits inside the iteration loop.
//   * compute: persistent CTAs of 128 threads pull tiles of unfrozen roots from an atomic counter.
//     A thread owns R roots (R = 2), and a root's sums are split over T threads (T = 1..128): the
//     T shares sit in different warps whenever T <= 4, so every shared-memory read of the pair loop
//     is a warp-wide broadcast and every value read is used for R roots.  Whole rounds of coarse
//     tiles are followed by fine tiles (4 T threads per root) that even out the last round.
//     Sources stream through shared memory in double-buffered stages of 256 stars + 512 roots,
//     each stage filled by three TMA bulk copies (cp.async.bulk) that complete on an mbarrier, so
//     no thread spends issue slots on loads.  One loop body evaluates one (root, star) pair in FP64
//     and two (root, root) pairs: the star sums carry F and must be FP64; the Aberth sum A only
//     steers the convergence RATE (it multiplies F in the denominator) and is evaluated in
//     double-single FP32 with packed f32x2 instructions, which read half the register-file bytes
//     of the FP64 form (register-operand bandwidth, one 64-bit operand per clock per SM
//     sub-partition, bounds this kernel: DESIGN.md "Measured issue model").
//   * Far-field mode: k_star_sums evaluates the star sums of every unfrozen root
//     from the near stars and the node's Taylor series (star_sums.cuh, fmm.cu); the compute kernel
//     then sums root pairs only (R = 8).
//   * Jacobi: updates go to a side buffer and are applied by the apply kernels, which also refresh the
//     per-slot source copy of the row and compact the list of unfrozen roots in order.
#include "star_sums.cuh"
#include "predictor.cuh"

#include <math.h>
#include <stdlib.h>
#include <algorithm>
#include <vector>

namespace mlcc {

// chain.cu: the small-field regime (one CTA per sub-chain)
struct ChainRun {
    unsigned long long root_iterations, root_iterations_noA;
    int max_iterations, unconverged_rows, degenerate;
};
int chain_capacity(int64_t N, int64_t n_r, bool caus);
int chain_launch(const double *star_xy, const double *masses, int64_t N, int64_t n_r, double gamma, double omk,
                 double tol, double skip_below, int max_iter, int max_iter_cold, int order, const void *d_rot,
                 const double *init_roots, double *roots, double *caustics, int *out_iters, int *out_unconverged,
                 int n_sub, const long long *d_first, const long long *d_centre, const long long *d_end,
                 void *d_counters, cudaStream_t stream);
size_t chain_counters_bytes();
void chain_read_counters(const void *h_counters, ChainRun *out);

namespace {

// Fields of up to this many roots per phase go to the chain regime when they fit it (mlcc_options.regime = AUTO);
// measured crossover: DESIGN.md "Kernel regimes".
constexpr int CHAIN_AUTO_MAX_ROOTS = 2400;

constexpr int CTA = 128;          // threads per CTA of the compute kernel
#ifndef MLCC_ROOTS_PER_THREAD
#define MLCC_ROOTS_PER_THREAD 2
#endif
#ifndef MLCC_MIN_CTAS
#define MLCC_MIN_CTAS 3
#endif
#ifndef MLCC_FINE_FACTOR
#define MLCC_FINE_FACTOR 4
#endif
constexpr int R_STARS = MLCC_ROOTS_PER_THREAD;   // roots per thread: every source read from shared memory is used R times
constexpr int R_ROOTS_F32 = 8;    // ... of the kernel that sums root pairs only (star sums from the node series)
constexpr int R_ROOTS_F64 = 4;
constexpr int S_TILE = 256;       // stars per stage; a stage also holds the 2*S_TILE roots paired with them
constexpr int STAGE_BYTES = S_TILE * 16 + S_TILE * 8 + 2 * S_TILE * 16;
constexpr int BLOCK = 256;        // threads per CTA of the small kernels
constexpr int MAX_ORDER = PRED_MAX_ORDER;      // highest predictor order
// Library default of the predictor's HIGHEST order (mlcc_options.predictor_order = -1); the order actually used is
// chosen root by root (predictor.cuh), so a high cap costs nothing where the history is rough or noisy.  Measured
// (R18): cfg4 5.47 / 5.01 / 4.94 / 4.92 s per set at caps 3 / 4 / 5 / 8, cfg5 25.1 / 22.4 / 21.7 s at 4 / 5 / 8.
constexpr int DEFAULT_ORDER_TILED = PRED_MAX_ORDER;
constexpr int DEFAULT_ORDER_CHAIN = PRED_MAX_ORDER;
constexpr int MAX_SLOTS = 1024;   // most slots in one step (2 per sub-chain)
constexpr double TINY = 1e-300;   // added to |d|^2 (FP64 root pairs): makes the self pair finite
constexpr float TINYF = 1e-30f;   // same for the FP32 root pairs
constexpr double PAD_STAR = 1e150;  // padding star: mass 0 at (1e150, 1e150); its 1/d ~ 1e-151 is lost in S1
constexpr float PAD_ROOT_F = 1e18f; // padding root of the FP32 source copy: its 1/d ~ 1e-18
constexpr int MODE_F32 = 0;       // Aberth sum in double-single FP32 (default)
constexpr int MODE_F64 = 1;       // Aberth sum in FP64 with the 20-bit reciprocal seed

// Tiles of one compute kernel.
struct TileSet {
    int T;                // threads per root in the coarse tiles
    int Tf;               // threads per root in the fine tiles (the last, partial round of work)
    int n_coarse;         // tiles [0, n_coarse) are coarse, [n_coarse, n_tiles) fine
    int n_tiles;
    int next_tile;        // tile counter of the running launch (atomic)
    int total;            // roots in these tiles
};

struct DevState {
    int step;             // newest step started: 0 = cold centre rows, s >= 1 = rows centre +/- s
    int iter;             // (unused)
    int n_slots;          // slot indices in use: gens * s2 (a slot with slot_step < 0 is free)
    int steps_final;      // every row of the steps below this one is final (no slot of theirs is live)
    int newest_roots;     // roots of the rows the newest step started with
    int done;             // all steps finished
    int need_seed;        // the seed kernel must write starting values for this step
    int cur;              // which of the two active lists is current
    TileSet ts[2];        // tiles of the next compute launches: [0] full kernel, [1] the one without the Aberth sum
    int total_active;     // unfrozen roots over all slots
    int total_iterations;
    int unconverged_rows;
    int degenerate;
    int n_outside;        // far-field mode: roots of this iteration that lie outside the node grid (atomic)
    long long root_iterations_noA;   // root-iterations done without the Aberth sum
    long long root_iterations;
    long long launches_used;  // compute launches that did work
};

struct Params {
    // problem
    const double2 *stars;     // [N]
    const double *masses;     // [N]
    int N;
    int n_r;                  // 2N
    int N_pad;                // N rounded up to a multiple of S_TILE
    double gamma;
    double mass0;             // masses[0]: the mass of every star in an equal-mass field (EQM kernels)
    double omk;               // 1 - kappa_s
    double tol2;              // tol^2
    int max_iter;
    int max_iter_cold;
    int order;                // predictor order
    int min_T;
    int grid_ctas;            // CTAs of the compute launch (all resident: one "round" = grid_ctas tiles)
    const double2 *rot;       // [num_phi]  (1-kappa_s) e^{-i phi_j}
    const double2 *init_roots;  // [n_r] or null
    double2 *roots;           // [num_phi][n_r]
    double2 *caustics;        // [num_phi][n_r] or null
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
    double2 *stars_pad;       // [N_pad]  stars, then padding stars
    double *mass_pad;         // [N_pad]
    float4 *src;              // [max_slots][2 N_pad] 16-byte source entries of the row each slot is solving:
                              //   MODE_F32: entries 2q, 2q+1 = (xh_a, xh_b, yh_a, yh_b), (xl_a, xl_b, yl_a, yl_b)
                              //             of roots a = 2q, b = 2q+1 (z = h + l, h = float(z), l = float(z - h))
                              //   MODE_F64: entry r = root r as double2
    long long *slot_row;      // [MAX_SLOTS] row solved by the slot in this step
    int *slot_sub;            // [MAX_SLOTS] sub-chain of the slot
    int *slot_dir;            // [MAX_SLOTS] -1, +1 (0 = centre)
    int *slot_iters;          // [MAX_SLOTS] iterations done on the slot's row
    int *slot_step;           // [MAX_SLOTS] step the slot's row belongs to, -1 = the slot is free
    int gens;                 // generations of slots that can be live at once (1 = lock-step)
    int s2;                   // slots per generation: 2 n_sub (sub-chain c: 2c downward / centre, 2c + 1 upward)
    int *n_active;            // [2][MAX_SLOTS]
    int *tile_start;          // [2 kernels][2][MAX_SLOTS + 1] first coarse / first fine tile of each slot
    int *coarse_roots;        // [2 kernels][MAX_SLOTS] roots of the slot covered by its coarse tiles
    int *n_small;             // [2][MAX_SLOTS] of the unfrozen roots of a slot, how many took a step below the
                              //   skip threshold last time: they sit at the END of the slot's list
    int *list;                // [2][max_slots][n_r]
    double2 *delta;           // [max_slots][n_r]
    int2 *chunk_count;        // [max_slots][chunks] survivors (with, without the Aberth sum) of every chunk of a slot's list
    unsigned *ticket;         // [1] CTAs of the running k_apply_write that are through
    int max_slots;            // slots that can be live at once (2 n_sub)
    int R;                    // roots per thread of the compute kernel in use
    // smooth-sheet polynomial H(u) = sum poly[n] u^n (rectangular field, Appendix B); poly_n = 0: none
    const double *poly;       // [poly_n] device
    int poly_n;
    double seed_radius;       // circle of the n_r - 2N extra cold seeds
    double skip_below2;       // a root whose last |Delta|^2 was below this is iterated without the Aberth sum; 0 = never
    int trust;                // mlcc_options.trust_predictor: rows seeded by the full-order predictor start without A
    // far-field mode (MLCC_STAR_SUMS_FMM): star sums come from k_star_sums, the compute kernel sums root pairs only
    double *ssum;             // [max_slots][n_r][8] star sums of the unfrozen roots, by list position
    int2 *outside;            // [max_slots * n_r] (slot, position) of the roots outside the node grid
    FmmGrid fmm;
};

// ------------------------------------------------------------------------------------------------
// small device helpers: packed FP32 arithmetic (FADD2 / FFMA2), mbarrier, TMA bulk copy
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 add2(float2 a, float2 b)
{
    float2 r;
    asm("{.reg .b64 ra, rb, rr; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; add.rn.ftz.f32x2 rr, ra, rb; "
        "mov.b64 {%0,%1}, rr;}" : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 sub2(float2 a, float2 b)
{
    float2 r;
    asm("{.reg .b64 ra, rb, rr; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; sub.rn.ftz.f32x2 rr, ra, rb; "
        "mov.b64 {%0,%1}, rr;}" : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c)
{
    float2 r;
    asm("{.reg .b64 ra, rb, rc, rr; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; mov.b64 rc, {%6,%7}; "
        "fma.rn.ftz.f32x2 rr, ra, rb, rc; mov.b64 {%0,%1}, rr;}"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return r;
}
__device__ __forceinline__ float rcp_f32(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ unsigned smem_u32(const void *p)
{
    return (unsigned)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    unsigned ok;
    do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!ok);
}
// TMA bulk copy global -> shared (bytes a multiple of 16, both addresses 16-byte aligned)
__device__ __forceinline__ void tma_load(void *dst, const void *src, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// double -> (h, l) with h = float(z), l = float(z - h): z = h + l to ~2^-48 relative
__device__ __forceinline__ void split_ds(double v, float &h, float &l)
{
    h = __double2float_rn(v);
    l = __double2float_rn(v - (double)h);
}

// writes root k of a slot's row into the slot's source copy
template <int MODE>
__device__ __forceinline__ void store_src(float4 *slot_src, int k, double2 z)
{
    if (MODE == MODE_F64) {
        reinterpret_cast<double2 *>(slot_src)[k] = z;
    } else {
        float xh, xl, yh, yl;
        split_ds(z.x, xh, xl);
        split_ds(z.y, yh, yl);
        float *f = reinterpret_cast<float *>(slot_src) + (size_t)(k >> 1) * 8 + (k & 1);
        f[0] = xh; f[2] = yh; f[4] = xl; f[6] = yl;
    }
}

// ------------------------------------------------------------------------------------------------
// pair bodies
// ------------------------------------------------------------------------------------------------
// (root, root) in FP64: A += 1/(z_k - z_r) with the 20-bit reciprocal seed.  Only the convergence
// RATE depends on A (the fixed point of the update is F = 0 whatever A is).  A root paired with
// itself has d = 0 exactly: |d|^2 + TINY = 1e-300, the seed is finite, the pair contributes 0.
__device__ __forceinline__ void pair_root_f64(double zx, double zy, double2 r, double &ax, double &ay)
{
    const double dx = zx - r.x;
    const double dy = r.y - zy;
    const double r2 = fma(dy, dy, fma(dx, dx, TINY));
    const double inv = rcp_seed(r2);
    ax = fma(dx, inv, ax);
    ay = fma(dy, inv, ay);
}

// two (root, root) pairs in double-single FP32, packed: lanes .x / .y of every float2 are the two
// source roots.  d = (zh - rh) + (zl - rl) is accurate to ~2^-23 |d| (the high parts cancel
// exactly when the roots are close), so 1/d carries ~6 digits like the FP64 seed form.
__device__ __forceinline__ void pair_root2_f32(float2 zxh, float2 zyh, float2 zxl, float2 zyl, float4 h, float4 l,
                                               float2 &ax, float2 &ay)
{
    const float2 dx = add2(sub2(zxh, make_float2(h.x, h.y)), sub2(zxl, make_float2(l.x, l.y)));
    const float2 dy = add2(sub2(make_float2(h.z, h.w), zyh), sub2(make_float2(l.z, l.w), zyl));
    const float2 r2 = fma2(dy, dy, fma2(dx, dx, make_float2(TINYF, TINYF)));
    const float2 inv = make_float2(rcp_f32(r2.x), rcp_f32(r2.y));
    ax = fma2(dx, inv, ax);
    ay = fma2(dy, inv, ay);
}

// ------------------------------------------------------------------------------------------------
// prepare kernel: padded star arrays, padding entries of every slot's source copy
// ------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void k_prepare(Params p)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    for (long long i = t0; i < p.N_pad; i += stride) {
        const bool real = i < p.N;
        p.stars_pad[i] = real ? p.stars[i] : make_double2(PAD_STAR, PAD_STAR);
        p.mass_pad[i] = real ? p.masses[i] : 0.0;
    }
    const int n_src = 2 * p.N_pad;
    const int n_padroots = n_src - p.n_r;
    for (long long idx = t0; idx < (long long)p.max_slots * n_padroots; idx += stride) {
        const int slot = (int)(idx / n_padroots);
        const int k = p.n_r + (int)(idx - (long long)slot * n_padroots);
        float4 *slot_src = p.src + (size_t)slot * n_src;
        if (MODE == MODE_F64) {
            reinterpret_cast<double2 *>(slot_src)[k] = make_double2(PAD_STAR, PAD_STAR);
        } else {
            float *f = reinterpret_cast<float *>(slot_src) + (size_t)(k >> 1) * 8 + (k & 1);
            f[0] = PAD_ROOT_F; f[2] = PAD_ROOT_F; f[4] = 0.f; f[6] = 0.f;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// seed kernel: starting values of every slot's new row + identity active lists
// ------------------------------------------------------------------------------------------------

template <int MODE>
__global__ void k_seed(Params p)
{
    const DevState st = *p.state;
    if (st.done || !st.need_seed) return;
    // the rows of the step that has just started sit in the slot block of its generation
    const int blk = (st.step % p.gens) * p.s2;
    const long long total = (long long)p.s2 * p.n_r;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int slot = blk + (int)(idx / p.n_r);
        const int k = (int)(idx - (long long)(slot - blk) * p.n_r);
        if (p.slot_step[slot] != st.step) continue;   // no row of this step in that slot
        const long long row = p.slot_row[slot];
        double2 z;
        if (st.step == 0) {
            if (p.init_roots) {
                z = p.init_roots[k];
            } else if (k < 2 * p.N) {  // z_i + 1, z_i - 1
                const int i = (k < p.N) ? k : k - p.N;
                z = p.stars[i];
                z.x += (k < p.N) ? 1.0 : -1.0;
            } else {  // "plus an additional number as required from alpha_s, evenly spread in a circle"
                double sn, cs;
                sincospi(2.0 * ((double)(k - 2 * p.N) + 0.5) / (double)(p.n_r - 2 * p.N), &sn, &cs);
                z = make_double2(p.seed_radius * cs, p.seed_radius * sn);
            }
        } else {
            // extrapolate through the last (order+1) rows of this chain that exist:
            // rows row - dir*q, q = 1 .. avail, lie inside the sub-chain and were solved in earlier steps
            const int sub = p.slot_sub[slot];
            const int dir = p.slot_dir[slot];
            long long room = (dir > 0) ? (row - p.sub_first[sub]) : (p.sub_end[sub] - 1 - row);
            long long avail = min((long long)(2 * st.step - 1), room);
            int order = (int)min((long long)p.order, avail - 1);
            double2 v[PRED_MAX_ORDER + 1];
#pragma unroll
            for (int q = 0; q <= PRED_MAX_ORDER; ++q)
                v[q] = q <= order ? p.roots[(row - (long long)dir * (q + 1)) * p.n_r + k] : make_double2(0.0, 0.0);
            z = predict_adaptive(v, order);
        }
        p.roots[row * p.n_r + k] = z;
        store_src<MODE>(p.src + (size_t)slot * 2 * p.N_pad, k, z);
        p.list[((long long)st.cur * p.max_slots + slot) * p.n_r + k] = k;
    }
}

// ------------------------------------------------------------------------------------------------
// compute kernel
// ------------------------------------------------------------------------------------------------
struct __align__(128) Stage {
    double2 sxy[S_TILE];     // star positions
    double sm[S_TILE];       // star masses
    float4 rp[2 * S_TILE];   // the slot's source entries 2 j0 .. 2 j0 + 2 S_TILE
};

// One Aberth step for the unfrozen root at position `pos` of the slot's list, from its sums:
//   t = 2 S1 - A,  S2 = (s2x, 2 s2h),  S3,  Sm (CAUS only).
template <bool CAUS>
__device__ __forceinline__ void aberth_step(const Params &p, int slot, long long row, const int *list, int pos,
                                            double tx, double ty, double s2x, double s2h, double s3x, double s3y,
                                            double smx, double smy)
{
    const int k = list[pos];
    const double2 z = p.roots[row * p.n_r + k];
    const double2 rot = p.rot[row];
    if (p.poly_n > 0) {
        // sheet polynomial with real coefficients: Sm += H(z), S2 -= H'(z), S3 += H''(z)/2, so that
        // F = gamma + S2 - (1-kappa_s) e^{-i phi}, F' = -2 S3 and the caustic expansion below hold as they are
        double b0x = 0, b0y = 0, b1x = 0, b1y = 0, b2x = 0, b2y = 0;
        for (int l = p.poly_n - 1; l >= 0; --l) {
            const double c = __ldg(&p.poly[l]);
            double tx_ = fma(b2x, z.x, fma(-b2y, z.y, b1x)), ty_ = fma(b2x, z.y, fma(b2y, z.x, b1y));
            b2x = tx_; b2y = ty_;
            tx_ = fma(b1x, z.x, fma(-b1y, z.y, b0x)); ty_ = fma(b1x, z.y, fma(b1y, z.x, b0y));
            b1x = tx_; b1y = ty_;
            tx_ = fma(b0x, z.x, fma(-b0y, z.y, c)); ty_ = fma(b0x, z.y, b0y * z.x);
            b0x = tx_; b0y = ty_;
        }
        smx += b0x; smy += b0y;
        s2x -= b1x; s2h -= 0.5 * b1y;
        s3x += b2x; s3y += b2y;
    }
    const double s2y = 2.0 * s2h;
    const double fx_ = p.gamma + s2x - rot.x;   // F
    const double fy_ = s2y - rot.y;
    const double gx = -2.0 * s3x;               // F'
    const double gy = -2.0 * s3y;
    const double dnx = gx + (fx_ * tx - fy_ * ty);  // F' + F (2 S1 - A)
    const double dny = gy + (fx_ * ty + fy_ * tx);
    const double dn2 = dnx * dnx + dny * dny;
    double2 d;
    d.x = (fx_ * dnx + fy_ * dny) / dn2;          // F / den
    d.y = (fy_ * dnx - fx_ * dny) / dn2;
    p.delta[(long long)slot * p.n_r + pos] = d;
    if (CAUS) {
        // caustic point of z' = z - Delta (Eq. 12) from the sums at z:
        // Sm(z') = Sm + Delta S2 + Delta^2 S3 + O(Delta^3 S4), Sm = sum m_i/(z - z_i);
        // exact to rounding once the root freezes (|Delta| < tol).  Rewritten every iteration.
        const double d2x = d.x * d.x - d.y * d.y, d2y = 2.0 * d.x * d.y;
        const double mx = smx + (d.x * s2x - d.y * s2y) + (d2x * s3x - d2y * s3y);
        const double my = smy + (d.x * s2y + d.y * s2x) + (d2x * s3y + d2y * s3x);
        const double nx = z.x - d.x, ny = z.y - d.y;
        double2 c;
        c.x = fma(p.omk + p.gamma, nx, -mx);   // (1-kappa_s) x + gamma x - Re Sm
        c.y = fma(p.omk - p.gamma, ny, my);    // (1-kappa_s) y - gamma y + Im Sm  (conj)
        p.caustics[row * p.n_r + k] = c;
    }
}

// Far-field mode: the star sums of every unfrozen root, one thread per root (near stars directly, distant
// stars from the node series: star_sums.cuh), written by list position for the compute kernel.
// grid: (ceil(n_r / BLOCK), max_slots)
__global__ void __launch_bounds__(BLOCK) k_star_sums(Params p)
{
    const DevState st = *p.state;
    if (st.done) return;
    const int slot = blockIdx.y;
    if (slot >= st.n_slots) return;
    const int n_act = p.n_active[st.cur * MAX_SLOTS + slot];
    const int pos = blockIdx.x * blockDim.x + threadIdx.x;
    if (pos >= n_act) return;
    const int *list = p.list + ((long long)st.cur * p.max_slots + slot) * p.n_r;
    const double2 z = p.roots[p.slot_row[slot] * p.n_r + list[pos]];
    StarAcc a = {0, 0, 0, 0, 0, 0, 0, 0};
    if (!fmm_star_sums(p.fmm, z.x, z.y, a)) {   // no node: queued for k_star_sums_outside
        p.outside[atomicAdd(&p.state->n_outside, 1)] = make_int2(slot, pos);
        return;
    }
    double2 *o = reinterpret_cast<double2 *>(p.ssum + ((size_t)slot * p.n_r + pos) * 8);
    o[0] = make_double2(a.s1x, a.s1y);
    o[1] = make_double2(a.s2x, a.s2h);
    o[2] = make_double2(a.s3x, a.s3y);
    o[3] = make_double2(a.smx, a.smy);
}

// The queued roots, one CTA per root: all stars directly, the CTA's shares added in a fixed tree.
__global__ void __launch_bounds__(BLOCK) k_star_sums_outside(Params p)
{
    __shared__ double s_red[BLOCK / 32][8];
    const DevState st = *p.state;
    if (st.done) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int q = blockIdx.x; q < st.n_outside; q += gridDim.x) {
        const int2 e = p.outside[q];
        const int *list = p.list + ((long long)st.cur * p.max_slots + e.x) * p.n_r;
        const double2 z = p.roots[p.slot_row[e.x] * p.n_r + list[e.y]];
        StarAcc a = {0, 0, 0, 0, 0, 0, 0, 0};
        for (int i = tid; i < p.N; i += BLOCK) pair_star<true>(z.x, z.y, p.stars[i], p.masses[i], a);
        double v[8] = {a.s1x, a.s1y, a.s2x, a.s2h, a.s3x, a.s3y, a.smx, a.smy};
#pragma unroll
        for (int c = 0; c < 8; ++c)
            for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
        __syncthreads();
        if (lane == 0) {
#pragma unroll
            for (int c = 0; c < 8; ++c) s_red[warp][c] = v[c];
        }
        __syncthreads();
        if (tid < 8) {
            double sum = 0.0;
            for (int w = 0; w < BLOCK / 32; ++w) sum += s_red[w][tid];
            p.ssum[((size_t)e.x * p.n_r + e.y) * 8 + tid] = sum;
        }
    }
}

// Thread layout of a tile with T threads per root: G = CTA / T threads share one value of `sub`
// (the share of the sources they sum: sources sub, sub + T, sub + 2T, ... of every stage) and
// thread (sub, local) owns the R roots at tile positions local, G + local, ...  For T <= CTA / 32
// a warp has ONE sub, so every shared-memory read in the pair loop is a warp-wide broadcast: a
// read costs the same wavefronts whatever T is, and each value read is used for R roots.
// STARS = false (far-field mode): the stages carry root entries only and the star sums are read
// from p.ssum; the loop body is then two packed FP32 root pairs per root, hence the larger R.
// ROOTS = false: the variant without the Aberth sum: the Newton step of F, t = 2 S1 - A left out as a whole, S1 not
// accumulated.  It takes the unfrozen roots whose last step was below
// the skip threshold (the tail [n_active - n_small, n_active) of every slot's list, tile set 1); the full kernel
// takes the others (tile set 0).  DESIGN.md readings R27, R30 (with trust_predictor: whole rows in their first iteration).
// EQM: every star has the mass p.mass0: the lighter pair body of star_sums.cuh (20 instead of 24 FP64 instructions).
template <int MODE, bool CAUS, bool STARS, bool ROOTS, int R, bool EQM = false>
__global__ void __launch_bounds__(CTA, STARS ? MLCC_MIN_CTAS : 4) k_compute(Params p)
{
    __shared__ Stage s_stage[2];
    __shared__ __align__(8) unsigned long long s_full[2];
    __shared__ int s_tile;
    constexpr int NV = STARS ? (CAUS ? 8 : 6) : 2;
    constexpr unsigned STAGE_TX = (STARS ? S_TILE * 24 : 0) + (ROOTS ? 2 * S_TILE * 16 : 0);
    constexpr bool STAGES = STARS || ROOTS;
    static_assert(sizeof(Stage) * 2 >= (size_t)NV * R * CTA * sizeof(double), "reduction scratch aliases the stages");

    const DevState st = *p.state;
    if (st.done) return;
    constexpr int K = ROOTS ? 0 : 1;
    const TileSet ts = st.ts[K];
    if (ts.n_tiles == 0) return;
    const int tid = threadIdx.x;
    const int n_stage = STAGES ? p.N_pad / S_TILE : 0;
    const int n_src = 2 * p.N_pad;
    // sources of the last stage that are not padding (a stage pairs star j with the root entries 2j, 2j + 1)
    const int last_cnt = max(p.N, (p.n_r + 1) / 2) - (n_stage - 1) * S_TILE;
    const int *n_active = p.n_active + st.cur * MAX_SLOTS;

    if (tid == 0) {
        mbar_init(&s_full[0], 1);
        mbar_init(&s_full[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    unsigned g = 0;   // stages consumed by this CTA so far: buffer g & 1, parity (g >> 1) & 1

    for (;;) {
        if (tid == 0) s_tile = atomicAdd(&p.state->ts[K].next_tile, 1);
        __syncthreads();
        const int tile = s_tile;
        if (tile >= ts.n_tiles) break;
        // coarse tiles first (whole rounds of the grid), then fine tiles (more threads per root, fewer
        // roots per tile) that even out the last, partial round
        const bool fine = tile >= ts.n_coarse;
        const int T = fine ? ts.Tf : ts.T;   // threads per root (power of two, 1..CTA)
        const int G = CTA / T;
        const int sub = tid / G;
        const int local = tid - sub * G;
        const int n_it = S_TILE / T;         // pair-loop iterations per stage (even, >= 2)
        const int n_it_last = min(n_it, ((last_cnt + T - 1) / T + 1) & ~1);   // the last stage stops at its padding
        const int tile_roots = R * G;
        const int *tab = p.tile_start + (2 * K + (fine ? 1 : 0)) * (MAX_SLOTS + 1);
        const int tt = fine ? tile - ts.n_coarse : tile;
        int lo = 0, hi = st.n_slots;         // slot of this tile: last slot with tab[slot] <= tt
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (tab[mid] <= tt) lo = mid; else hi = mid;
        }
        const int slot = lo;
        const long long row = p.slot_row[slot];
        const float4 *slot_src = p.src + (size_t)slot * n_src;
        // Tiles whose roots are spread over the WHOLE CTA (T = CTA: the straggler iterations of a step, a handful of
        // unfrozen roots) read their sources straight from global memory (L2): every thread has only N_pad / CTA
        // sources, so the staged pipeline would be a chain of n_stage copy latencies (43 us per launch at N = 10^4)
        // with nothing to overlap them; independent loads take a few microseconds.
        const bool direct = STAGES && T == CTA;
        if (STAGES && !direct && tid == 0) {   // first stage of this tile
            const unsigned b = g & 1u;
            mbar_expect_tx(&s_full[b], STAGE_TX);
            if (STARS) {
                tma_load(s_stage[b].sxy, p.stars_pad, S_TILE * 16, &s_full[b]);
                tma_load(s_stage[b].sm, p.mass_pad, S_TILE * 8, &s_full[b]);
            }
            if (ROOTS) tma_load(s_stage[b].rp, slot_src, 2 * S_TILE * 16, &s_full[b]);
        }
        const int *list = p.list + ((long long)st.cur * p.max_slots + slot) * p.n_r;
        // this kernel's share of the slot's list: positions [pos_lo, n_act)
        const int n_all = n_active[slot], n_large = n_all - p.n_small[st.cur * MAX_SLOTS + slot];
        const int pos_lo = ROOTS ? 0 : n_large;
        const int n_act = ROOTS ? n_large : n_all;
        const int base = pos_lo + (fine ? p.coarse_roots[K * MAX_SLOTS + slot] : 0) + (tt - tab[slot]) * tile_roots;
        const bool valid = base + local < n_act;   // this thread has at least its first root
        double zx[R], zy[R];
        float zxh[R], zxl[R], zyh[R], zyl[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            // a thread whose r-th position is past the end repeats its first root (result dropped)
            const int pos = base + r * G + local;
            const int pp = pos < n_act ? pos : base + local;
            double2 z = make_double2(0.0, 0.0);
            if (valid) z = p.roots[row * p.n_r + list[pp]];
            zx[r] = z.x;
            zy[r] = z.y;
            split_ds(z.x, zxh[r], zxl[r]);
            split_ds(z.y, zyh[r], zyl[r]);
        }
        StarAcc acc[STARS ? R : 1];
        double ax[R], ay[R], bx[R], by[R];   // MODE_F64: two chains
        float2 fx[R], fy[R];                 // MODE_F32: packed lanes
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (STARS) acc[r] = StarAcc{0, 0, 0, 0, 0, 0, 0, 0};
            ax[r] = ay[r] = bx[r] = by[r] = 0.0;
            fx[r] = fy[r] = make_float2(0.f, 0.f);
        }

        for (int t = 0; t < (direct ? 0 : n_stage); ++t, ++g) {
            const unsigned b = g & 1u;
            if (tid == 0 && t + 1 < n_stage) {   // prefetch: buffer b^1 was last read in stage g-1, closed by a barrier
                const unsigned nb = b ^ 1u;
                mbar_expect_tx(&s_full[nb], STAGE_TX);
                if (STARS) {
                    tma_load(s_stage[nb].sxy, p.stars_pad + (size_t)(t + 1) * S_TILE, S_TILE * 16, &s_full[nb]);
                    tma_load(s_stage[nb].sm, p.mass_pad + (size_t)(t + 1) * S_TILE, S_TILE * 8, &s_full[nb]);
                }
                if (ROOTS) tma_load(s_stage[nb].rp, slot_src + (size_t)(t + 1) * 2 * S_TILE, 2 * S_TILE * 16, &s_full[nb]);
            }
            mbar_wait(&s_full[b], (g >> 1) & 1u);
            if (valid) {
                const Stage &sg = s_stage[b];
                // blocks of 2 sources x R roots: independent (1 star + 2 roots) bodies with no exit in
                // between, so that their dependent chains (|d|^2 -> reciprocal -> powers) interleave
                // (the packed-FP32 variant keeps the fixed trip count: with the variable one its loop came out 4.6 %
                // slower per pair on sm_100a, more than the 2.4 % of padding pairs it would save at cfg4)
                const int n_it_t = (MODE == MODE_F32 || t + 1 < n_stage) ? n_it : n_it_last;
                for (int i = 0; i < n_it_t; i += 2) {
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        const int j = sub + (i + u) * T;
                        double2 sxy = make_double2(0.0, 0.0);
                        double sm = 0.0;
                        if (STARS) {
                            sxy = sg.sxy[j];
                            if (!EQM) sm = sg.sm[j];
                        }
                        if (!ROOTS) {
#pragma unroll
                            for (int r = 0; r < R; ++r)
                                if (STARS) {
                                    if (EQM) pair_star_eq<CAUS, false>(zx[r], zy[r], sxy, acc[r]);
                                    else pair_star<CAUS, false>(zx[r], zy[r], sxy, sm, acc[r]);
                                }
                        } else if (MODE == MODE_F64) {
                            const double2 *rr = reinterpret_cast<const double2 *>(sg.rp);
                            const double2 ra = rr[2 * j], rb = rr[2 * j + 1];
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                if (STARS) {
                                    if (EQM) pair_star_eq<CAUS>(zx[r], zy[r], sxy, acc[r]);
                                    else pair_star<CAUS>(zx[r], zy[r], sxy, sm, acc[r]);
                                }
                                pair_root_f64(zx[r], zy[r], ra, ax[r], ay[r]);
                                pair_root_f64(zx[r], zy[r], rb, bx[r], by[r]);
                            }
                        } else {
                            const float4 h = sg.rp[2 * j], l = sg.rp[2 * j + 1];
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                if (STARS) {
                                    if (EQM) pair_star_eq<CAUS>(zx[r], zy[r], sxy, acc[r]);
                                    else pair_star<CAUS>(zx[r], zy[r], sxy, sm, acc[r]);
                                }
                                pair_root2_f32(make_float2(zxh[r], zxh[r]), make_float2(zyh[r], zyh[r]),
                                               make_float2(zxl[r], zxl[r]), make_float2(zyl[r], zyl[r]), h, l,
                                               fx[r], fy[r]);
                            }
                        }
                    }
                }
            }
            __syncthreads();   // everyone is done with buffer b before it is refilled
        }
        if (direct && valid) {
            // thread `tid` takes the sources tid, tid + CTA, ... (star j with the root entries 2j, 2j + 1, as a stage
            // pairs them); N_pad is a multiple of 2 CTA
#pragma unroll 2
            for (int j0 = tid; j0 < p.N_pad; j0 += 2 * CTA) {
                double2 sxy[2];
                double sm[2];
                float4 e0[2], e1[2];
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    const int j = j0 + u * CTA;
                    sxy[u] = make_double2(0.0, 0.0);
                    sm[u] = 0.0;
                    e0[u] = e1[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (STARS) {
                        sxy[u] = __ldg(&p.stars_pad[j]);
                        if (!EQM) sm[u] = __ldg(&p.mass_pad[j]);
                    }
                    if (ROOTS) {
                        e0[u] = __ldg(&slot_src[2 * j]);
                        e1[u] = __ldg(&slot_src[2 * j + 1]);
                    }
                }
#pragma unroll
                for (int u = 0; u < 2; ++u) {
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        if (STARS) {
                            if (EQM) pair_star_eq<CAUS, ROOTS>(zx[r], zy[r], sxy[u], acc[r]);
                            else pair_star<CAUS, ROOTS>(zx[r], zy[r], sxy[u], sm[u], acc[r]);
                        }
                        if (ROOTS && MODE == MODE_F64) {
                            const double2 ra = make_double2(__hiloint2double(__float_as_int(e0[u].y), __float_as_int(e0[u].x)),
                                                            __hiloint2double(__float_as_int(e0[u].w), __float_as_int(e0[u].z)));
                            const double2 rb = make_double2(__hiloint2double(__float_as_int(e1[u].y), __float_as_int(e1[u].x)),
                                                            __hiloint2double(__float_as_int(e1[u].w), __float_as_int(e1[u].z)));
                            pair_root_f64(zx[r], zy[r], ra, ax[r], ay[r]);
                            pair_root_f64(zx[r], zy[r], rb, bx[r], by[r]);
                        } else if (ROOTS) {
                            pair_root2_f32(make_float2(zxh[r], zxh[r]), make_float2(zyh[r], zyh[r]),
                                           make_float2(zxl[r], zxl[r]), make_float2(zyl[r], zyl[r]), e0[u], e1[u],
                                           fx[r], fy[r]);
                        }
                    }
                }
            }
        }
        // ---- this thread's partial sums: v = (2 S1 - A, S2, S3, Sm), or (-A) alone without STARS ----
        double v[R][NV];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            double sax, say;
            if (MODE == MODE_F32) {
                sax = (double)fx[r].x + (double)fx[r].y;
                say = (double)fy[r].x + (double)fy[r].y;
            } else {
                sax = ax[r] + bx[r];
                say = ay[r] + by[r];
            }
            if (STARS && EQM) star_sums_scale<CAUS, ROOTS>(acc[r], p.mass0);
            if (STARS) {
                // without the Aberth sum the step is the Newton step of F: t = 2 S1 - A is left out as a whole
                // (2 S1 and A nearly cancel -- two roots per star -- so 2 S1 alone would be the worse stand-in)
                v[r][0] = ROOTS ? 2.0 * acc[r].s1x - sax : 0.0;
                v[r][1] = ROOTS ? 2.0 * acc[r].s1y - say : 0.0;
                v[r][2] = acc[r].s2x; v[r][3] = acc[r].s2h; v[r][4] = acc[r].s3x; v[r][5] = acc[r].s3y;
                if (CAUS) { v[r][NV - 2] = acc[r].smx; v[r][NV - 1] = acc[r].smy; }
            } else {
                v[r][0] = -sax;
                v[r][1] = -say;
            }
        }
        // the step of the root at list position `pos` from its combined sums w[0..NV)
        auto finish = [&](int pos, const double *w) {
            if (STARS) {
                aberth_step<CAUS>(p, slot, row, list, pos, w[0], w[1], w[2], w[3], w[4], w[5],
                                  CAUS ? w[NV - 2] : 0.0, CAUS ? w[NV - 1] : 0.0);
            } else {
                const double2 *s = reinterpret_cast<const double2 *>(p.ssum + ((size_t)slot * p.n_r + pos) * 8);
                const double2 s1 = s[0], s2 = s[1], s3 = s[2], smm = s[3];
                aberth_step<CAUS>(p, slot, row, list, pos, ROOTS ? fma(2.0, s1.x, w[0]) : 0.0,
                                  ROOTS ? fma(2.0, s1.y, w[1]) : 0.0, s2.x, s2.y, s3.x, s3.y, smm.x, smm.y);
            }
        };
        if (T == 1) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int pos = base + r * G + local;
                if (pos < n_act) finish(pos, v[r]);
            }
        } else {
            // combine the T shares through shared memory (the stage buffers are idle: every stage of
            // this tile has been consumed and the next tile's first copy is issued after the barrier below)
            double *red = reinterpret_cast<double *>(s_stage);   // [NV][T][tile_roots]
#pragma unroll
            for (int r = 0; r < R; ++r)
#pragma unroll
                for (int q = 0; q < NV; ++q) red[(q * T + sub) * tile_roots + r * G + local] = v[r][q];
            __syncthreads();
            for (int e = tid; e < tile_roots && base + e < n_act; e += CTA) {   // tile_roots > CTA when T < R
                double w[NV];
#pragma unroll
                for (int q = 0; q < NV; ++q) {
                    double sum = 0.0;
                    for (int s2 = 0; s2 < T; ++s2) sum += red[(q * T + s2) * tile_roots + e];
                    w[q] = sum;
                }
                finish(base + e, w);
            }
            // order these generic-proxy accesses before the async-proxy (TMA) writes of the next tile
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        }
        __syncthreads();   // s_tile and the stage buffers are rewritten by the next tile
    }
}

// ------------------------------------------------------------------------------------------------
// helpers of the apply kernels (below, after the state machine they end in)
// ------------------------------------------------------------------------------------------------
// mlcc_options.trust_predictor (R30): the rows of a step whose seeds come from the predictor at its
// full order start with every root in the no-Aberth-sum group; k_apply guards that first iteration.
__device__ __forceinline__ bool trusted_step(const Params &p, int step)
{
    return p.trust && p.skip_below2 > 0.0 && p.order >= 1 && step >= 1 && 2 * step - 1 >= p.order + 1;
}

// What becomes of a root after a finite step of squared size d2 (both passes of k_apply use this one predicate):
//   0 frozen (|Delta| < tol), 1 "large": iterated next with the Aberth sum, 2 "small": iterated next without it.
// guard = first iteration of a trusted row (the steps were Newton steps from predicted seeds): a step of at least
// the skip threshold is REJECTED -- kind 1 whatever tol is, z unchanged -- and a smaller one is applied.
__device__ __forceinline__ int step_kind(double d2, double tol2, double skip2, bool guard)
{
    if (guard && !(d2 < skip2)) return 1;
    if (d2 < tol2) return 0;
    return d2 < skip2 ? 2 : 1;
}

// ------------------------------------------------------------------------------------------------
// state machine (k_init, finalize_iteration): one CTA of FIN threads, thread s looks after slot s
// (MAX_SLOTS = FIN), sums and prefix sums over the slots by block-wide scans
// ------------------------------------------------------------------------------------------------
constexpr int FIN = MAX_SLOTS;

// exclusive prefix sum of v over the CTA's threads; *total = the sum (the same value in every thread)
__device__ __forceinline__ long long block_scan(long long v, long long *total, long long *s_buf /*[33]*/)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    long long incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const long long t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    __syncthreads();   // s_buf may still be read from the previous call
    if (lane == 31) s_buf[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        const long long w = s_buf[lane];
        long long wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const long long t = __shfl_up_sync(0xffffffffu, wi, o);
            if (lane >= o) wi += t;
        }
        s_buf[lane] = wi - w;
        if (lane == 31) s_buf[32] = wi;
    }
    __syncthreads();
    *total = s_buf[32];
    return s_buf[warp] + incl - v;
}

// The tile table of the next compute launch for the counts in n_active[cur].
// All grid_ctas CTAs are resident and pull tiles from one atomic counter, and tiles of one kind take the
// same time, so a launch lasts ceil(tiles / grid_ctas) tile-times: with a handful of tiles per CTA
// the last, partial round costs up to a whole round.  Hence two kinds of tile:
//   coarse: T threads per root, R CTA / T roots per tile, T the smallest power of two that gives at
//           least two rounds; only WHOLE rounds of them are handed out;
//   fine:   Tf = MLCC_FINE_FACTOR T threads per root for what is left of every slot's list, so the
//           partial round is quantised in units of 1 / MLCC_FINE_FACTOR of a coarse tile.
// Every thread returns with the same st.
__device__ void build_tiles_of(const Params &p, DevState &st, int K, int count, long long *s_buf)
{
    // count = this slot's roots for kernel K (0 for the threads beyond n_slots)
    const int s = threadIdx.x;
    long long total, W, tc_total, tf_total;
    block_scan(count, &total, s_buf);
    int T = 1;
    while (T < CTA && total * T / (p.R * CTA) < 2LL * p.grid_ctas) T <<= 1;
    if (T < p.min_T) T = p.min_T;
    int Tf = T * MLCC_FINE_FACTOR;
    if (Tf > CTA) Tf = CTA;
    const int tile_c = p.R * CTA / T, tile_f = p.R * CTA / Tf;
    block_scan(count / tile_c, &W, s_buf);   // coarse tiles if every slot were cut into coarse tiles only
    const long long C = (W / p.grid_ctas) * p.grid_ctas;   // whole rounds
    const int c_s = (W > 0 && Tf != T) ? (int)((long long)(count / tile_c) * C / W) : 0;
    const int f_s = (count - c_s * tile_c + tile_f - 1) / tile_f;
    const long long tc = block_scan(c_s, &tc_total, s_buf);
    const long long tf = block_scan(f_s, &tf_total, s_buf);
    int *tab_c = p.tile_start + (2 * K) * (MAX_SLOTS + 1), *tab_f = tab_c + MAX_SLOTS + 1;
    if (s < st.n_slots) {
        tab_c[s] = (int)tc;
        tab_f[s] = (int)tf;
        p.coarse_roots[K * MAX_SLOTS + s] = c_s * tile_c;
    }
    if (s == 0) {
        tab_c[st.n_slots] = (int)tc_total;
        tab_f[st.n_slots] = (int)tf_total;
    }
    TileSet &ts = st.ts[K];
    ts.T = T;
    ts.Tf = Tf;
    ts.n_coarse = (int)tc_total;
    ts.n_tiles = (int)(tc_total + tf_total);
    ts.next_tile = 0;
    ts.total = (int)total;
}

// both kernels' tile sets for the counts in n_active[cur] / n_small[cur]
__device__ void build_tiles(const Params &p, DevState &st, long long *s_buf)
{
    const int s = threadIdx.x;
    const int n_act = s < st.n_slots ? __ldcg(&p.n_active[st.cur * MAX_SLOTS + s]) : 0;
    const int n_sm = s < st.n_slots ? __ldcg(&p.n_small[st.cur * MAX_SLOTS + s]) : 0;
    build_tiles_of(p, st, 0, n_act - n_sm, s_buf);
    build_tiles_of(p, st, 1, n_sm, s_buf);
    st.total_active = st.ts[0].total + st.ts[1].total;
}

// Starts step st.step: thread c looks after sub-chain c (n_sub <= MAX_SLOTS / 2).  The rows of the step take the
// slot block of the step's generation, (st.step % gens) * s2 + {2c: downward (or the centre row), 2c + 1: upward};
// st.cur is the list the next launches read.  Every thread returns with the same st.
__device__ void spawn_step(const Params &p, DevState &st, long long *s_buf)
{
    const int c = threadIdx.x;
    int has_dn = 0, has_up = 0;
    long long row_dn = 0, row_up = 0;
    if (c < p.n_sub) {
        if (st.step == 0) {
            has_dn = 1;                      // the centre row, direction 0
            row_dn = p.sub_centre[c];
        } else {
            row_up = p.sub_centre[c] + st.step;
            row_dn = p.sub_centre[c] - st.step;
            has_dn = row_dn >= p.sub_first[c];
            has_up = row_up < p.sub_end[c];
        }
    }
    const int blk = (st.step % p.gens) * p.s2;
    // a new row: every root gets the Aberth sum, unless the step's seeds are trusted (then none does at first)
    const int n_small0 = trusted_step(p, st.step) ? p.n_r : 0;
    for (int q = 0; q < 2; ++q) {
        if (!(q == 0 ? has_dn : has_up)) continue;
        const int slot = blk + 2 * c + q;
        p.slot_row[slot] = q == 0 ? row_dn : row_up;
        p.slot_sub[slot] = c;
        p.slot_dir[slot] = q == 0 ? (st.step == 0 ? 0 : -1) : +1;
        p.slot_step[slot] = st.step;
        p.slot_iters[slot] = 0;
        p.n_active[st.cur * MAX_SLOTS + slot] = p.n_r;
        p.n_active[(st.cur ^ 1) * MAX_SLOTS + slot] = 0;
        p.n_small[st.cur * MAX_SLOTS + slot] = n_small0;
        p.n_small[(st.cur ^ 1) * MAX_SLOTS + slot] = 0;
    }
    long long n;
    block_scan(has_dn + has_up, &n, s_buf);
    st.newest_roots = (int)(n * p.n_r);
    st.need_seed = 1;
    __syncthreads();   // the counts are read back by build_tiles
}

// input check: flags[0] = non-finite star coordinates / masses, flags[1] = pairs of coincident stars
// (two stars at the same point make P(z) lose two roots: the degree claim 2N fails),
// flags[2] = masses that differ from masses[0] (0: an equal-mass field, which takes the lighter pair body)
__global__ void k_check_stars(const double2 *__restrict__ stars, const double *__restrict__ masses, int N,
                              int *flags)
{
    __shared__ double2 s_xy[BLOCK];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double2 me = make_double2(0.0, 0.0);
    if (i < N) {
        me = stars[i];
        const double m = masses[i];
        if (!(fabs(me.x) <= 1e100) || !(fabs(me.y) <= 1e100) || !(fabs(m) <= 1e100)) atomicAdd(&flags[0], 1);
        if (m != masses[0]) atomicAdd(&flags[2], 1);
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

__global__ void __launch_bounds__(FIN) k_init(Params p)
{
    __shared__ long long s_buf[33];
    DevState st;
    st.step = 0; st.iter = 0; st.n_slots = p.gens * p.s2; st.done = 0; st.need_seed = 1; st.cur = 0;
    st.steps_final = 0; st.newest_roots = 0;
    st.ts[0] = TileSet{1, 1, 0, 0, 0, 0}; st.ts[1] = TileSet{1, 1, 0, 0, 0, 0};
    st.total_active = 0; st.total_iterations = 0;
    st.unconverged_rows = 0; st.degenerate = 0; st.n_outside = 0; st.root_iterations_noA = 0; st.root_iterations = 0; st.launches_used = 0;
    p.slot_step[threadIdx.x] = -1;   // FIN = MAX_SLOTS threads: every slot free (n_active / n_small were zeroed by the host)
    __syncthreads();
    spawn_step(p, st, s_buf);
    build_tiles(p, st, s_buf);
    if (threadIdx.x == 0) *p.state = st;
}

// Closes an iteration (run by the LAST CTA of k_apply_write, FIN threads).  Every live slot has been iterated once:
// a slot whose list is empty (or that has used up its iterations) is finished -- its row's diagnostics are written
// and the slot is freed; the next step is STARTED as soon as (a) the slot block of its generation is free and (b) the
// newest step has almost no survivor with a large step left (at most one root in 1024; the cold step must be
// finished altogether): the few roots of older rows that still need iterations are carried along as extra slots of
// the same launches instead of holding up the whole step.  A row seeded from a predecessor that
// is still moving by < 1e-8 gets a seed that is off by as much: only the starting guess sees it.
__device__ void finalize_iteration(const Params &p, long long *s_buf)
{
    DevState st = *p.state;   // every thread carries the same copy and makes the same decisions
    if (st.done) return;
    const int s = threadIdx.x;
    // the iteration that just ran
    st.total_iterations += 1;
    st.root_iterations += st.total_active;
    st.root_iterations_noA += st.ts[1].total;
    st.launches_used += 1;
    st.need_seed = 0;
    st.n_outside = 0;
    int my_step = -1, unconv = 0, large = 0;
    if (s < st.n_slots && (my_step = p.slot_step[s]) >= 0) {
        const int it = p.slot_iters[s] + 1;
        p.slot_iters[s] = it;
        // (written by other CTAs of this launch: read through L2)
        const int left = __ldcg(&p.n_active[(st.cur ^ 1) * MAX_SLOTS + s]);
        const int cap = (my_step == 0) ? p.max_iter_cold : p.max_iter;
        if (left == 0 || it >= cap) {            // the row is finished
            const long long row = p.slot_row[s];
            if (p.out_iters) p.out_iters[row] = it;
            if (p.out_unconverged) p.out_unconverged[row] = left;
            if (left > 0) {
                unconv = 1;
                p.n_active[(st.cur ^ 1) * MAX_SLOTS + s] = 0;
                p.n_small[(st.cur ^ 1) * MAX_SLOTS + s] = 0;
            }
            p.slot_step[s] = -1;
            my_step = -1;
        } else if (my_step == st.step) {
            large = left - __ldcg(&p.n_small[(st.cur ^ 1) * MAX_SLOTS + s]);
        }
    }
    // live slots per generation (step - g, g = 0 .. gens - 1 <= 2) in 16-bit fields, unconverged rows above them
    long long packed = (long long)unconv << 48;
    if (my_step >= 0) packed += 1ll << (16 * (st.step - my_step));
    long long tot_packed, tot_large;
    block_scan(packed, &tot_packed, s_buf);
    block_scan(large, &tot_large, s_buf);
    st.unconverged_rows += (int)(tot_packed >> 48);
    const int live_g[3] = {(int)(tot_packed & 0xffff), (int)((tot_packed >> 16) & 0xffff), (int)((tot_packed >> 32) & 0xffff)};
    const int live_total = live_g[0] + live_g[1] + live_g[2];
    st.cur ^= 1;
    st.steps_final = st.step + 1;
    for (int g = 0; g < p.gens; ++g)
        if (live_g[g] > 0) st.steps_final = st.step - g;
    bool spawn = false;
    if (st.step < p.max_steps) {
        const bool block_free = live_g[p.gens - 1] == 0;   // the slot block of step + 1 is that of step + 1 - gens
        const bool newest_ok = st.step == 0 ? live_total == 0 : tot_large <= (long long)(st.newest_roots >> 10);
        spawn = block_free && newest_ok;
    }
    if (spawn) {
        st.step += 1;
        spawn_step(p, st, s_buf);
    } else if (st.step >= p.max_steps && live_total == 0) {
        st.done = 1;
    }
    if (!st.done) build_tiles(p, st, s_buf);
    __syncthreads();   // every thread has read *p.state
    if (s == 0) *p.state = st;
}

// ------------------------------------------------------------------------------------------------
// apply: z_k -= Delta_k, freeze converged roots, compact the list of unfrozen roots IN ORDER (survivors that keep the
// Aberth sum first, then the others), so the next iteration's tiles -- and with them the summation order of every
// root -- do not depend on the timing of a launch: two runs give the same bits.
// A slot's list is cut into chunks of APPLY_CHUNK entries, one CTA each:
//   k_apply_count  counts the two kinds of survivors of every chunk (reads the steps only);
//   k_apply_write  applies the steps and writes the survivors at the offsets the counts give; the last CTA of the
//                  grid to finish (a ticket) then closes the iteration (finalize_iteration).
// grid of both: (chunks of the longest list, max_slots)
// ------------------------------------------------------------------------------------------------
constexpr int APPLY_THREADS = FIN;   // the last CTA runs the state machine: one thread per slot
constexpr int APPLY_ITEMS = 4;
constexpr int APPLY_CHUNK = APPLY_THREADS * APPLY_ITEMS;
constexpr int COUNT_THREADS = 256;

__global__ void __launch_bounds__(COUNT_THREADS) k_apply_count(Params p)
{
    __shared__ int s_part[2][COUNT_THREADS / 32];
    const DevState st = *p.state;
    if (st.done) return;
    const int slot = blockIdx.y, chunk = blockIdx.x;
    if (slot >= st.n_slots) return;
    const int n_act = p.n_active[st.cur * MAX_SLOTS + slot];
    const int lo = chunk * APPLY_CHUNK, hi = min(n_act, lo + APPLY_CHUNK);
    if (lo >= n_act) return;
    const double2 *delta = p.delta + (long long)slot * p.n_r;
    const bool guard = p.slot_iters[slot] == 0 && trusted_step(p, p.slot_step[slot]);
    int n_large = 0, n_small = 0;
    for (int pos = lo + threadIdx.x; pos < hi; pos += COUNT_THREADS) {
        const double2 d = delta[pos];
        const double d2 = d.x * d.x + d.y * d.y;
        if (d2 <= 1.79769313486231570e308) {
            const int kind = step_kind(d2, p.tol2, p.skip_below2, guard);
            n_large += kind == 1;
            n_small += kind == 2;
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        n_large += __shfl_xor_sync(0xffffffffu, n_large, o);
        n_small += __shfl_xor_sync(0xffffffffu, n_small, o);
    }
    if ((threadIdx.x & 31) == 0) { s_part[0][threadIdx.x >> 5] = n_large; s_part[1][threadIdx.x >> 5] = n_small; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int a = 0, b = 0;
        for (int w = 0; w < COUNT_THREADS / 32; ++w) { a += s_part[0][w]; b += s_part[1][w]; }
        p.chunk_count[(size_t)slot * gridDim.x + chunk] = make_int2(a, b);
    }
}

template <int MODE>
__global__ void __launch_bounds__(APPLY_THREADS) k_apply_write(Params p)
{
    __shared__ int s_warp[32];
    __shared__ int s_total;
    __shared__ long long s_buf[33];
    __shared__ int s_last;
    const DevState st = *p.state;
    if (st.done) return;
    const int slot = blockIdx.y, chunk = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_act = slot < st.n_slots ? p.n_active[st.cur * MAX_SLOTS + slot] : 0;
    const int c0 = chunk * APPLY_CHUNK;
    if (c0 < n_act || (chunk == 0 && slot < st.n_slots)) {
        // offsets of this chunk from the counts of the slot's chunks: large survivors first, then the small ones
        const int n_chunks = (n_act + APPLY_CHUNK - 1) / APPLY_CHUNK;
        int base_l = 0, base_s = 0, tot_l = 0, tot_s = 0;
        for (int c = 0; c < n_chunks; ++c) {
            const int2 v = p.chunk_count[(size_t)slot * gridDim.x + c];
            if (c < chunk) { base_l += v.x; base_s += v.y; }
            tot_l += v.x;
            tot_s += v.y;
        }
        base_s += tot_l;
        if (chunk == 0 && tid == 0) {
            p.n_active[(st.cur ^ 1) * MAX_SLOTS + slot] = tot_l + tot_s;
            p.n_small[(st.cur ^ 1) * MAX_SLOTS + slot] = tot_s;
        }
        if (c0 < n_act) {
            const int *list = p.list + ((long long)st.cur * p.max_slots + slot) * p.n_r;
            int *next = p.list + ((long long)(st.cur ^ 1) * p.max_slots + slot) * p.n_r;
            const double2 *delta = p.delta + (long long)slot * p.n_r;
            double2 *row = p.roots + p.slot_row[slot] * p.n_r;
            float4 *slot_src = p.src + (size_t)slot * 2 * p.N_pad;
            // First iteration of a trusted row: the steps were taken without the Aberth sum, i.e. they are Newton steps
            // from the predicted seeds.  One below the skip threshold is applied as any confirming step is; a larger one
            // says the prediction was not that good: it is NOT applied and the root gets a full Aberth iteration next.
            const bool guard = p.slot_iters[slot] == 0 && trusted_step(p, p.slot_step[slot]);
            int ks[APPLY_ITEMS];
            int kind[APPLY_ITEMS];   // 0 frozen, 1 large, 2 small
            int cnt = 0;
#pragma unroll
            for (int i = 0; i < APPLY_ITEMS; ++i) {
                const int pos = c0 + tid * APPLY_ITEMS + i;
                kind[i] = 0;
                ks[i] = 0;
                if (pos < n_act) {
                    const int k = list[pos];
                    const double2 d = delta[pos];
                    const double d2 = d.x * d.x + d.y * d.y;
                    if (d2 <= 1.79769313486231570e308) {   // finite step
                        kind[i] = step_kind(d2, p.tol2, p.skip_below2, guard);
                        if (!(guard && kind[i] == 1)) {     // (a rejected Newton step leaves z where it is)
                            double2 z = row[k];
                            z.x -= d.x;
                            z.y -= d.y;
                            row[k] = z;
                            store_src<MODE>(slot_src, k, z);
                        }
                    } else {                                // NaN / Inf: freeze where it is, report
                        atomicAdd(&p.state->degenerate, 1);
                    }
                    ks[i] = k;
                    cnt += kind[i] == 1 ? 1 : (kind[i] == 2 ? (1 << 16) : 0);
                }
            }
            int incl = cnt;   // inclusive scan over the warp, then over the warps (counts packed: large low, small high)
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int n = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += n;
            }
            if (lane == 31) s_warp[warp] = incl;
            __syncthreads();
            if (warp == 0) {
                const int w = s_warp[lane];
                int wi = w;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int n = __shfl_up_sync(0xffffffffu, wi, o);
                    if (lane >= o) wi += n;
                }
                s_warp[lane] = wi - w;
                if (lane == 31) s_total = wi;
            }
            __syncthreads();
            const int excl = s_warp[warp] + incl - cnt;
            int off_l = base_l + (excl & 0xffff), off_s = base_s + (excl >> 16);
#pragma unroll
            for (int i = 0; i < APPLY_ITEMS; ++i) {
                if (kind[i] == 1) next[off_l++] = ks[i];
                else if (kind[i] == 2) next[off_s++] = ks[i];
            }
        }
    }
    // ---- the last CTA to get here closes the iteration ----
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        const unsigned total = gridDim.x * gridDim.y;
        const unsigned t = atomicAdd(p.ticket, 1u);
        s_last = (t == total - 1);
        if (s_last) *p.ticket = 0;   // for the next launch (ordered by the stream)
    }
    __syncthreads();
    if (s_last) {
        __threadfence();
        finalize_iteration(p, s_buf);
    }
}

// the kernels of one Aberth-sum mode / caustic fusion choice
struct KernelSet {
    void (*prepare)(Params);
    void (*seed)(Params);
    void (*compute)(Params);
    void (*compute_noA)(Params);   // the variant without the Aberth sum, for the roots whose last step was small
    void (*apply)(Params);
    int R;   // roots per thread of `compute`
};

template <int MODE>
KernelSet kernel_set_mode(bool caus, bool fmm, bool eqm)
{
    constexpr int RR = MODE == MODE_F64 ? R_ROOTS_F64 : R_ROOTS_F32;
    KernelSet k;
    k.prepare = k_prepare<MODE>; k.seed = k_seed<MODE>; k.apply = k_apply_write<MODE>;
    if (fmm) {
        k.compute = caus ? k_compute<MODE, true, false, true, RR> : k_compute<MODE, false, false, true, RR>;
        k.compute_noA = caus ? k_compute<MODE, true, false, false, RR> : k_compute<MODE, false, false, false, RR>;
        k.R = RR;
    } else if (eqm) {
        k.compute = caus ? k_compute<MODE, true, true, true, R_STARS, true> : k_compute<MODE, false, true, true, R_STARS, true>;
        k.compute_noA = caus ? k_compute<MODE, true, true, false, R_STARS, true> : k_compute<MODE, false, true, false, R_STARS, true>;
        k.R = R_STARS;
    } else {
        k.compute = caus ? k_compute<MODE, true, true, true, R_STARS> : k_compute<MODE, false, true, true, R_STARS>;
        k.compute_noA = caus ? k_compute<MODE, true, true, false, R_STARS> : k_compute<MODE, false, true, false, R_STARS>;
        k.R = R_STARS;
    }
    return k;
}

KernelSet kernel_set(int mode, bool caus, bool fmm, bool eqm)
{
    return mode == MODE_F64 ? kernel_set_mode<MODE_F64>(caus, fmm, eqm) : kernel_set_mode<MODE_F32>(caus, fmm, eqm);
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
        // enough slots (2 per sub-chain) to keep ~4.8e5 roots in flight, but chains at least 16 rows long.  More rows
        // per step mean fewer steps, and every step ends with two or three launches for a handful of straggler roots
        // (~80 us each, whatever the field); more sub-chains mean more cold rows (~7.6 full row-iterations each).
        // Measured on B200, seconds per curve set at 3e5 / 4.8e5 / 6.4e5 / 9.6e5 roots in flight: cfg4 4.919 / 4.855 /
        // 4.856 / 4.882, cfg3 0.1175 / 0.1162 / 0.1188 / 0.1250.
        const int64_t n_r = 2 * N;
        int64_t slots = (480000 + n_r - 1) / n_r;
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

// The iteration groups are replayed from a CUDA graph (below), and stream capture is not allowed on the legacy
// default stream: a call on that stream runs on a library-owned stream instead, ordered after the caller's stream by
// an event at the start; the call synchronises before it returns, which orders it before whatever follows.
struct RunStream {
    cudaStream_t run = nullptr;
    bool owned = false;
    cudaError_t open(cudaStream_t caller)
    {
        run = caller;
        if (caller != nullptr && caller != cudaStreamLegacy) return cudaSuccess;
        cudaStream_t s = nullptr;
        cudaError_t e = cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking);
        if (e != cudaSuccess) return e;
        cudaEvent_t ready = nullptr;
        e = cudaEventCreateWithFlags(&ready, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventRecord(ready, caller);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s, ready, 0);
        if (ready) cudaEventDestroy(ready);
        if (e != cudaSuccess) { cudaStreamDestroy(s); return e; }
        run = s;
        owned = true;
        return cudaSuccess;
    }
    ~RunStream()
    {
        if (owned) { cudaStreamSynchronize(run); cudaStreamDestroy(run); }
    }
};

// The chain regime: stars checked, one launch, one read-back (flags + counters), rows copied to the host buffers
// of the _host entry points at the end (these fields are small).
static int chain_solve(const double *star_xy, const double *masses, int64_t N, int n_r, double kappa_s, double gamma,
                       int64_t num_phi, double tol, double skip_below, int max_iter, int max_iter_cold, int order,
                       const std::vector<double2> &rot, int n_sub, const std::vector<long long> &first,
                       const std::vector<long long> &centre, const std::vector<long long> &end, int max_steps,
                       const double *init_roots, double *out_roots, double *out_caustics, int32_t *out_iters,
                       int32_t *out_unconverged, mlcc_stats *out_stats, cudaStream_t stream, double *h_roots,
                       double *h_caustics)
{
    NvtxRange nvtx_("mlcc: solve, chain regime (star check + one launch: cold rows and continuation steps run on chip)");
    Workspace ws(stream);
    double2 *d_rot = nullptr;
    long long *d_plan = nullptr;
    int *d_flags = nullptr;
    unsigned char *d_counters = nullptr;
    const size_t cbytes = chain_counters_bytes();
    MLCC_CUDA(ws.alloc(&d_rot, (size_t)num_phi));
    MLCC_CUDA(ws.alloc(&d_plan, (size_t)3 * n_sub));
    MLCC_CUDA(ws.alloc(&d_flags, 4));
    MLCC_CUDA(ws.alloc(&d_counters, cbytes));
    static thread_local PinnedBlock tl_back;   // flags + counters come back through pinned memory
    MLCC_CUDA(tl_back.reserve(2 * sizeof(int) + 8 + cbytes));
    int *h_flags = static_cast<int *>(tl_back.p);
    unsigned char *h_counters = static_cast<unsigned char *>(tl_back.p) + 16;
    std::vector<long long> plan((size_t)3 * n_sub);
    for (int c = 0; c < n_sub; ++c) { plan[c] = first[c]; plan[n_sub + c] = centre[c]; plan[2 * n_sub + c] = end[c]; }
    MLCC_CUDA(cudaMemcpyAsync(d_rot, rot.data(), sizeof(double2) * (size_t)num_phi, cudaMemcpyHostToDevice, stream));
    MLCC_CUDA(cudaMemcpyAsync(d_plan, plan.data(), sizeof(long long) * plan.size(), cudaMemcpyHostToDevice, stream));
    MLCC_CUDA(cudaMemsetAsync(d_flags, 0, 4 * sizeof(int), stream));
    Event ev0, ev1;
    MLCC_CUDA(ev0.create());
    MLCC_CUDA(ev1.create());
    MLCC_CUDA(cudaEventRecord(ev0, stream));
    k_check_stars<<<(unsigned)((N + BLOCK - 1) / BLOCK), BLOCK, 0, stream>>>(
        reinterpret_cast<const double2 *>(star_xy), masses, (int)N, d_flags);
    const int lrc = chain_launch(star_xy, masses, N, n_r, gamma, 1.0 - kappa_s, tol, skip_below, max_iter, max_iter_cold,
                                 order, d_rot, init_roots, out_roots, out_caustics, out_iters, out_unconverged, n_sub,
                                 d_plan, d_plan + n_sub, d_plan + 2 * n_sub, d_counters, stream);
    if (lrc != MLCC_OK) return lrc;
    MLCC_CUDA(cudaEventRecord(ev1, stream));
    MLCC_CUDA(cudaMemcpyAsync(h_flags, d_flags, 2 * sizeof(int), cudaMemcpyDeviceToHost, stream));
    MLCC_CUDA(cudaMemcpyAsync(h_counters, d_counters, cbytes, cudaMemcpyDeviceToHost, stream));
    if (h_roots) {
        const size_t bytes = (size_t)num_phi * n_r * 2 * sizeof(double);
        MLCC_CUDA(cudaMemcpyAsync(h_roots, out_roots, bytes, cudaMemcpyDeviceToHost, stream));
        if (h_caustics && out_caustics)
            MLCC_CUDA(cudaMemcpyAsync(h_caustics, out_caustics, bytes, cudaMemcpyDeviceToHost, stream));
    }
    cudaError_t es = cudaStreamSynchronize(stream);
    if (es == cudaSuccess) es = cudaGetLastError();
    if (es != cudaSuccess) return cuda_fail(es, "critical-curve kernel (chain regime)", __FILE__, __LINE__);
    if (h_flags[0]) return invalid("non-finite (or > 1e100) star position or mass");
    if (h_flags[1]) {
        set_last_error("coincident stars: P(z) loses roots (merge them into one star of the summed mass)");
        return MLCC_ERR_DEGENERATE;
    }
    ChainRun run{};
    chain_read_counters(h_counters, &run);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, ev0, ev1);
    if (out_stats) {
        out_stats->root_iterations = (int64_t)run.root_iterations;
        out_stats->star_pairs = (int64_t)run.root_iterations * N;
        out_stats->root_pairs = (int64_t)(run.root_iterations - run.root_iterations_noA) * (n_r - 1);
        out_stats->kernel_launches = 2;   // star check, chain kernel
        out_stats->total_iterations = run.max_iterations;   // the longest CTA's iterations: the critical path
        out_stats->steps = max_steps + 1;
        out_stats->subchains = n_sub;
        out_stats->predictor_order = order;
        out_stats->unconverged_rows = run.unconverged_rows;
        out_stats->degenerate_roots = run.degenerate;
        out_stats->solve_ms = ms;
        out_stats->aberth_sum_precision = 64;
        out_stats->regime = MLCC_REGIME_CHAIN;
    }
    if (run.degenerate > 0) {
        set_last_error("NaN/Inf Aberth step: a root landed on a star or another root, or stars coincide");
        return MLCC_ERR_DEGENERATE;
    }
    if (run.unconverged_rows > 0) {
        set_last_error("some roots were still unfrozen at max_iter");
        return MLCC_ERR_NOT_CONVERGED;
    }
    return MLCC_OK;
}

// h_roots / h_caustics (host-buffer entry points; may be null): PINNED host arrays of the shape of out_roots /
// out_caustics.  Rows are final as soon as their step is over (nothing writes them again, the predictor only reads
// them) and a sub-chain's finished rows are one interval that grows at both ends, so the rows each poll of the state
// reports finished are copied device -> host on a second, non-blocking stream while the solve goes on: the 16 bytes
// per root and per caustic point of the output cross PCIe under the kernels instead of after them.
int critical_curves_impl(const double *star_xy, const double *masses, int64_t N, double kappa_s,
                         double gamma, int64_t num_phi, double tol, int32_t max_iter,
                         double *out_roots, double *out_caustics, const mlcc_options *opt_in,
                         const double *init_roots, int32_t *out_iters, int32_t *out_unconverged,
                         mlcc_stats *out_stats, cudaStream_t stream, double *h_roots, double *h_caustics)
{
    if (!star_xy || !masses || !out_roots) return invalid("null pointer");
    if (N < 1 || N > (1 << 28)) return invalid("N out of range");
    if (num_phi < 1) return invalid("num_phi < 1");
    if (!(tol > 0.0) || !isfinite(tol)) return invalid("tol must be positive and finite");
    if (max_iter < 1) return invalid("max_iter < 1");
    if (!isfinite(kappa_s) || !isfinite(gamma)) return invalid("kappa_s / gamma not finite");
    if (out_caustics == out_roots) return invalid("out_caustics aliases out_roots");
    mlcc_options opt;
    mlcc_options_default(&opt);
    if (opt_in) {
        if (opt_in->struct_size != 0 && opt_in->struct_size != (int32_t)sizeof(mlcc_options))
            return invalid("mlcc_options.struct_size");
        opt = *opt_in;
    }
    const int64_t phi_total = opt.phi_index_total > 0 ? opt.phi_index_total : num_phi;
    const int64_t phi_off = opt.phi_index_offset;
    int order = opt.predictor_order < 0 ? DEFAULT_ORDER_TILED : opt.predictor_order;
    if (order > MAX_ORDER) return invalid("predictor_order > 8");
    int min_T = opt.min_lanes_per_root <= 0 ? 1 : opt.min_lanes_per_root;
    if (min_T > CTA || (min_T & (min_T - 1))) return invalid("min_lanes_per_root must be a power of two <= 128");
    if (opt.num_subchains < 0 || opt.max_iter_cold < 0) return invalid("negative option");
    if (opt.aberth_sum_precision != 0 && opt.aberth_sum_precision != 32 && opt.aberth_sum_precision != 64)
        return invalid("aberth_sum_precision must be 0, 32 or 64");
    const int mode = opt.aberth_sum_precision == 32 ? MODE_F32 : MODE_F64;   // 0 = library default = FP64
    if (opt.regime != MLCC_REGIME_AUTO && opt.regime != MLCC_REGIME_TILED && opt.regime != MLCC_REGIME_CHAIN)
        return invalid("regime");
    if (!isfinite(opt.skip_aberth_sum_below)) return invalid("skip_aberth_sum_below");
    if (opt.trust_predictor != 0 && opt.trust_predictor != 1) return invalid("trust_predictor must be 0 or 1");
    if (opt.star_sum_mode != MLCC_STAR_SUMS_DIRECT && opt.star_sum_mode != MLCC_STAR_SUMS_FMM)
        return invalid("star_sum_mode");

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

    // sheet polynomial: n_extra = deg H' = poly_n - 2 more roots per row
    const int poly_n = opt.sheet_poly ? opt.sheet_poly_n : 0;
    if (poly_n < 0 || poly_n > 512) return invalid("sheet_poly_n out of range");
    if (poly_n > 0) {
        for (int q = 0; q < poly_n; ++q)
            if (!isfinite(opt.sheet_poly[q])) return invalid("sheet_poly has a non-finite coefficient");
        if (opt.sheet_poly[poly_n - 1] == 0.0) return invalid("the last sheet_poly coefficient is zero");
    }
    const int n_extra = poly_n >= 3 ? poly_n - 2 : 0;
    if (n_extra > 0 && !init_roots && !(opt.seed_radius > 0.0 && isfinite(opt.seed_radius)))
        return invalid("seed_radius must be positive when the sheet polynomial adds roots");
    if (2 * N + n_extra > (1ll << 30)) return invalid("too many roots");
    const int n_r = (int)(2 * N) + n_extra;
    // a stage pairs 256 stars with 512 root entries: enough (massless, far away) padding stars for all roots
    const long long n_half = (n_r + 1) / 2 > N ? (n_r + 1) / 2 : N;
    const int N_pad = (int)((n_half + S_TILE - 1) / S_TILE) * S_TILE;

    // ---- which regime ----
    // chain: one CTA per sub-chain, everything in shared memory (chain.cu); tiled: the launches below.
    const bool use_fmm = opt.star_sum_mode == MLCC_STAR_SUMS_FMM;
    const bool chain_able = !use_fmm && poly_n == 0 && opt.trust_predictor == 0 && opt.aberth_sum_precision != 32 &&
                            opt.min_lanes_per_root <= 1;
    int chain_cap = 0;
    if (opt.regime != MLCC_REGIME_TILED && chain_able) chain_cap = chain_capacity(N, n_r, out_caustics != nullptr);
    if (opt.regime == MLCC_REGIME_CHAIN && chain_cap < 1)
        return invalid("regime = MLCC_REGIME_CHAIN needs direct star sums, no sheet polynomial, no trust_predictor, "
                       "an FP64 Aberth sum and a field that fits shared memory (about 1200 stars)");
    const bool use_chain = chain_cap >= 1 && (opt.regime == MLCC_REGIME_CHAIN || n_r <= CHAIN_AUTO_MAX_ROOTS);

    // plan
    std::vector<long long> first(MAX_SLOTS), centre(MAX_SLOTS), end(MAX_SLOTS);
    std::vector<int64_t> f64v(MAX_SLOTS), c64v(MAX_SLOTS), e64v(MAX_SLOTS);
    int want_sub = opt.num_subchains;
    if (want_sub == 0 && use_chain) {
        // one CTA per sub-chain, one wave of CTAs; a cold row costs about as much as two continued ones, so chains
        // shorter than 8 rows are not worth their cold start
        long long w = std::min<long long>(chain_cap, num_phi / 8);
        want_sub = (int)std::max<long long>(1, std::min<long long>(w, MAX_SLOTS / 2));
    }
    if (want_sub == 0 && opt.trust_predictor == 1 && opt.star_sum_mode == MLCC_STAR_SUMS_FMM) {
        // Continued rows cost O(N) here (far-field star sums, no Aberth sum): a step of the default plan is a handful
        // of short, latency-bound launches.  More rows per step amortise them; the price is as many more cold rows
        // (measured on cfg4: 0.53 s per set with 8 sub-chains, 0.34 s with 32; 2.5 times the default plan is 30).
        const int base = plan_subchains_host(N, num_phi, 0, MAX_SLOTS / 2, f64v.data(), c64v.data(), e64v.data());
        if (base >= 1) {
            long long w = 5ll * base / 2;
            if (w > num_phi / 16) w = num_phi / 16;
            if (w > MAX_SLOTS / 2) w = MAX_SLOTS / 2;
            want_sub = (int)(w > base ? w : base);
        }
    }
    const int n_sub = plan_subchains_host(N, num_phi, want_sub, MAX_SLOTS / 2, f64v.data(),
                                          c64v.data(), e64v.data());
    if (n_sub < 1) return invalid("num_subchains");
    int max_steps = 0;
    for (int c = 0; c < n_sub; ++c) {
        first[c] = f64v[c]; centre[c] = c64v[c]; end[c] = e64v[c];
        const long long a = centre[c] - first[c], b = end[c] - 1 - centre[c];
        if (a > max_steps) max_steps = (int)a;
        if (b > max_steps) max_steps = (int)b;
    }
    const int order_used = opt.predictor_order < 0 ? DEFAULT_ORDER_CHAIN : opt.predictor_order;
    if (use_chain) {
        const double sb = opt.skip_aberth_sum_below == 0.0 ? 1e-8 : opt.skip_aberth_sum_below;   // on at every N here
        return chain_solve(star_xy, masses, N, n_r, kappa_s, gamma, num_phi, tol, sb, max_iter,
                           opt.max_iter_cold > 0 ? opt.max_iter_cold : max_iter, order_used, rot, n_sub, first, centre,
                           end, max_steps, init_roots, out_roots, out_caustics, out_iters, out_unconverged, out_stats,
                           stream, h_roots, h_caustics);
    }
    // up to three generations of slots live at once: the rows of the newest step, and what is left of the two before
    const int s2 = 2 * n_sub;
    int gens = 3;
    while (gens > 1 && gens * s2 > MAX_SLOTS) --gens;
    const int max_slots = gens * s2;
    NvtxRange nvtx_("mlcc: solve, tiled regime");
    RunStream run_stream;            // declared before the workspace: destroyed after it
    MLCC_CUDA(run_stream.open(stream));
    stream = run_stream.run;
    Workspace ws(stream);
    Params p{};
    double2 *d_rot = nullptr;
    long long *d_plan = nullptr;
    cudaError_t e;
    if ((e = ws.alloc(&d_rot, (size_t)num_phi)) != cudaSuccess ||
        (e = ws.alloc(&d_plan, (size_t)3 * n_sub)) != cudaSuccess ||
        (e = ws.alloc(&p.state, 1)) != cudaSuccess ||
        (e = ws.alloc(&p.stars_pad, (size_t)N_pad)) != cudaSuccess ||
        (e = ws.alloc(&p.mass_pad, (size_t)N_pad)) != cudaSuccess ||
        (e = ws.alloc(&p.src, (size_t)max_slots * 2 * N_pad)) != cudaSuccess ||
        (e = ws.alloc(&p.slot_row, MAX_SLOTS)) != cudaSuccess ||
        (e = ws.alloc(&p.slot_sub, MAX_SLOTS)) != cudaSuccess ||
        (e = ws.alloc(&p.slot_dir, MAX_SLOTS)) != cudaSuccess ||
        (e = ws.alloc(&p.slot_iters, MAX_SLOTS)) != cudaSuccess ||
        (e = ws.alloc(&p.slot_step, MAX_SLOTS)) != cudaSuccess ||
        (e = ws.alloc(&p.n_active, 2 * MAX_SLOTS)) != cudaSuccess ||
        (e = ws.alloc(&p.tile_start, 4 * (MAX_SLOTS + 1))) != cudaSuccess ||
        (e = ws.alloc(&p.coarse_roots, 2 * MAX_SLOTS)) != cudaSuccess ||
        (e = ws.alloc(&p.n_small, 2 * MAX_SLOTS)) != cudaSuccess ||
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
    MLCC_CUDA(cudaMemsetAsync(p.n_small, 0, sizeof(int) * 2 * MAX_SLOTS, stream));

    // input check (one small read-back before the solve); flags[2] = 0 says every star has the mass masses[0]
    int h_flags[3] = {0, 0, 0};
    double mass0 = 0.0;
    {
        int *d_flags = nullptr;
        MLCC_CUDA(ws.alloc(&d_flags, 4));
        MLCC_CUDA(cudaMemsetAsync(d_flags, 0, 4 * sizeof(int), stream));
        k_check_stars<<<(unsigned)((N + BLOCK - 1) / BLOCK), BLOCK, 0, stream>>>(
            reinterpret_cast<const double2 *>(star_xy), masses, (int)N, d_flags);
        MLCC_CUDA(cudaMemcpyAsync(h_flags, d_flags, 3 * sizeof(int), cudaMemcpyDeviceToHost, stream));
        MLCC_CUDA(cudaMemcpyAsync(&mass0, masses, sizeof(double), cudaMemcpyDeviceToHost, stream));
        MLCC_CUDA(cudaStreamSynchronize(stream));
        MLCC_CUDA(cudaGetLastError());
        if (h_flags[0]) return invalid("non-finite (or > 1e100) star position or mass");
        if (h_flags[1]) {
            set_last_error("coincident stars: P(z) loses roots (merge them into one star of the summed mass)");
            return MLCC_ERR_DEGENERATE;
        }
    }

    const bool eqm = h_flags[2] == 0;
    const KernelSet ks = kernel_set(mode, out_caustics != nullptr, use_fmm, eqm);
    int blocks_per_sm = 0;
    MLCC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks_per_sm, ks.compute, CTA, 0));
    if (blocks_per_sm < 1) blocks_per_sm = 1;
    const int sms = device_sm_count();
    const int grid_compute = sms * blocks_per_sm;

    p.stars = reinterpret_cast<const double2 *>(star_xy);
    p.masses = masses;
    p.N = (int)N;
    p.n_r = n_r;
    p.N_pad = N_pad;
    p.gamma = gamma;
    p.mass0 = mass0;
    p.omk = 1.0 - kappa_s;
    p.tol2 = tol * tol;
    p.max_iter = max_iter;
    p.max_iter_cold = opt.max_iter_cold > 0 ? opt.max_iter_cold : max_iter;
    p.order = order;
    p.min_T = min_T;
    p.grid_ctas = grid_compute;
    p.R = ks.R;
    const double skip_below = opt.skip_aberth_sum_below == 0.0 ? 1e-8 : opt.skip_aberth_sum_below;
    // The second compute launch per iteration pays off where the Aberth sum is the bulk of the work.  Small fields are
    // launch bound (cfg1: 2.7 ms per curve set with it, 2.0 ms without): there it is used only if asked for by
    // an explicit threshold or by trust_predictor.
    const bool skip_on = skip_below > 0.0 &&
                         (N >= 512 || opt.skip_aberth_sum_below > 0.0 || opt.trust_predictor != 0);
    p.skip_below2 = skip_on ? skip_below * skip_below : 0.0;
    p.trust = opt.trust_predictor != 0 ? 1 : 0;
    p.poly_n = poly_n;
    p.seed_radius = opt.seed_radius;
    if (poly_n > 0) {
        double *d_poly = nullptr;
        MLCC_CUDA(ws.alloc(&d_poly, (size_t)poly_n));
        MLCC_CUDA(cudaMemcpyAsync(d_poly, opt.sheet_poly, sizeof(double) * poly_n, cudaMemcpyHostToDevice, stream));
        p.poly = d_poly;
    }
    p.rot = d_rot;
    p.init_roots = reinterpret_cast<const double2 *>(init_roots);
    p.roots = reinterpret_cast<double2 *>(out_roots);
    p.caustics = reinterpret_cast<double2 *>(out_caustics);
    p.out_iters = out_iters;
    p.out_unconverged = out_unconverged;
    p.n_sub = n_sub;
    p.sub_first = d_plan;
    p.sub_centre = d_plan + n_sub;
    p.sub_end = d_plan + 2 * n_sub;
    p.max_steps = max_steps;
    p.max_slots = max_slots;
    p.gens = gens;
    p.s2 = s2;

    Event ev0, ev1, ev_poll[2];
    MLCC_CUDA(ev0.create());
    MLCC_CUDA(ev1.create());
    MLCC_CUDA(ev_poll[0].create(cudaEventDisableTiming));
    MLCC_CUDA(ev_poll[1].create(cudaEventDisableTiming));
    // pinned, two snapshots of the device state, kept per host thread (PinnedBlock)
    static thread_local PinnedBlock tl_state;
    MLCC_CUDA(tl_state.reserve(2 * sizeof(DevState)));
    DevState *h_state = static_cast<DevState *>(tl_state.p);
    h_state[0].done = h_state[1].done = 0;

    MLCC_CUDA(cudaEventRecord(ev0, stream));
    int64_t launches = 3;   // check, prepare, init
    if (use_fmm) {   // grid + node series of the far field, once per call (inside the timed region)
        MLCC_CUDA(ws.alloc(&p.ssum, (size_t)max_slots * n_r * 8));
        MLCC_CUDA(ws.alloc(&p.outside, (size_t)max_slots * n_r));
        const int frc = fmm_build(p.stars, masses, (int)N, opt.fmm_order, opt.fmm_stars_per_node, ws, &p.fmm, stream);
        if (frc != MLCC_OK) return frc;
        launches += 9;
    }
    const int grid_seed = sms * 4;
    ks.prepare<<<grid_seed, BLOCK, 0, stream>>>(p);
    k_init<<<1, FIN, 0, stream>>>(p);
    const int n_chunks = (n_r + APPLY_CHUNK - 1) / APPLY_CHUNK;
    const dim3 grid_apply((unsigned)n_chunks, (unsigned)max_slots);
    MLCC_CUDA(ws.alloc(&p.chunk_count, (size_t)n_chunks * max_slots));
    MLCC_CUDA(ws.alloc(&p.ticket, 1));
    MLCC_CUDA(cudaMemsetAsync(p.ticket, 0, sizeof(unsigned), stream));
    const dim3 grid_star((unsigned)((n_r + BLOCK - 1) / BLOCK), (unsigned)max_slots);
    // Upper bound on iteration groups, so that a device-side fault cannot spin the host forever.
    const long long max_groups = (long long)(max_steps + 1) * (long long)(p.max_iter > p.max_iter_cold ? p.max_iter : p.max_iter_cold) + 8;
    const int chunk = 16;
    long long groups = 0;
    int which = 0;
    bool finished = false;
    int rc = MLCC_OK;
    // progressive copy of finished rows to the host (see the comment above the function)
    OwnedStream copy_stream;
    std::vector<long long> c_lo(n_sub, 0), c_hi(n_sub, -1);   // rows of sub-chain c already handed to the copy stream
    if (h_roots) MLCC_CUDA(copy_stream.create());
    auto copy_rows = [&](long long a, long long b) {
        if (a > b) return;
        const size_t off = (size_t)a * n_r * 2, bytes = (size_t)(b - a + 1) * n_r * 2 * sizeof(double);
        cudaMemcpyAsync(h_roots + off, out_roots + off, bytes, cudaMemcpyDeviceToHost, copy_stream);
        if (h_caustics && out_caustics)
            cudaMemcpyAsync(h_caustics + off, out_caustics + off, bytes, cudaMemcpyDeviceToHost, copy_stream);
    };
    // the rows solved in steps < steps_final are final: row centre +- q, q < steps_final, inside the sub-chain
    auto copy_finished = [&](long long steps_final) {
        if (!h_roots || steps_final < 1) return;
        for (int c = 0; c < n_sub; ++c) {
            const long long lo = std::max(first[c], centre[c] - (steps_final - 1));
            const long long hi = std::min(end[c] - 1, centre[c] + (steps_final - 1));
            if (c_lo[c] > c_hi[c]) copy_rows(lo, hi);
            else { copy_rows(lo, c_lo[c] - 1); copy_rows(c_hi[c] + 1, hi); }
            c_lo[c] = lo; c_hi[c] = hi;
        }
    };
    auto enqueue_chunk = [&]() {
        for (int g = 0; g < chunk; ++g) {
            ks.seed<<<grid_seed, BLOCK, 0, stream>>>(p);
            if (use_fmm) {
                k_star_sums<<<grid_star, BLOCK, 0, stream>>>(p);
                k_star_sums_outside<<<sms, BLOCK, 0, stream>>>(p);
            }
            ks.compute<<<grid_compute, CTA, 0, stream>>>(p);
            if (skip_on) ks.compute_noA<<<grid_compute, CTA, 0, stream>>>(p);
            k_apply_count<<<grid_apply, COUNT_THREADS, 0, stream>>>(p);
            ks.apply<<<grid_apply, APPLY_THREADS, 0, stream>>>(p);
        }
    };
    // Every launch of a chunk has the same arguments (the state lives on the device), so the chunk is captured once
    // and replayed: small fields are pure launch latency (cfg1: ~8 us per launch from the host).  Any failure of the
    // capture falls back to plain launches.
    cudaGraphExec_t chunk_exec = nullptr;
    {
        // kernels are loaded lazily at their first launch, and loading is not allowed inside a capture: touch them first
        cudaFuncAttributes fa;
        const void *fns[] = {(const void *)ks.seed, (const void *)ks.compute, (const void *)ks.compute_noA,
                             (const void *)ks.apply, (const void *)k_apply_count, (const void *)k_star_sums,
                             (const void *)k_star_sums_outside};
        for (const void *f : fns) cudaFuncGetAttributes(&fa, f);
        cudaGetLastError();
        cudaGraph_t graph = nullptr;
        if (cudaStreamBeginCapture(stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            enqueue_chunk();
            if (cudaStreamEndCapture(stream, &graph) == cudaSuccess && graph) {
                if (cudaGraphInstantiate(&chunk_exec, graph, 0) != cudaSuccess) chunk_exec = nullptr;
            }
            if (graph) cudaGraphDestroy(graph);
        }
        if (!chunk_exec) cudaGetLastError();
    }
    int steps_seen = 0;
    while (!finished && groups < max_groups + 2 * chunk) {
        NvtxRange nvtx_chunk("mlcc: enqueue a chunk of 16 iteration groups (seed, compute, apply)");
        if (!chunk_exec || cudaGraphLaunch(chunk_exec, stream) != cudaSuccess) {
            if (chunk_exec) { cudaGetLastError(); cudaGraphExecDestroy(chunk_exec); chunk_exec = nullptr; }
            enqueue_chunk();
        }
        launches += ((use_fmm ? 6 : 4) + (skip_on ? 1 : 0)) * chunk;
        groups += chunk;
        cudaMemcpyAsync(&h_state[which], p.state, sizeof(DevState), cudaMemcpyDeviceToHost, stream);
        cudaEventRecord(ev_poll[which], stream);
        // look at the previous chunk's snapshot while this one runs
        if (groups > chunk) {
            cudaError_t es = cudaEventSynchronize(ev_poll[which ^ 1]);
            if (es != cudaSuccess) { rc = cuda_fail(es, "cudaEventSynchronize", __FILE__, __LINE__); break; }
            if (h_state[which ^ 1].done) finished = true;
            if (h_state[which ^ 1].steps_final > steps_seen) {   // step 0 = the cold centre rows, then the continuation steps
                char text[96];
                snprintf(text, sizeof text, "mlcc: steps %d..%d finished (step 0 = cold rows)", steps_seen,
                         h_state[which ^ 1].steps_final - 1);
                nvtxMarkA(text);
                steps_seen = h_state[which ^ 1].steps_final;
            }
            copy_finished(h_state[which ^ 1].steps_final);   // that snapshot is complete: every launch before it has run
        }
        which ^= 1;
    }
    if (chunk_exec) cudaGraphExecDestroy(chunk_exec);
    DevState fin{};
    if (rc == MLCC_OK) {
        cudaEventRecord(ev1, stream);
        cudaError_t es = cudaMemcpyAsync(&h_state[0], p.state, sizeof(DevState), cudaMemcpyDeviceToHost, stream);
        if (es == cudaSuccess) es = cudaStreamSynchronize(stream);
        if (es == cudaSuccess) es = cudaGetLastError();
        if (es != cudaSuccess) rc = cuda_fail(es, "critical-curve kernels", __FILE__, __LINE__);
        else fin = h_state[0];
    }
    if (copy_stream.s) {
        if (rc == MLCC_OK && fin.done) copy_finished((long long)max_steps + 1);   // whatever is left
        cudaError_t es = cudaStreamSynchronize(copy_stream);
        if (rc == MLCC_OK && es != cudaSuccess) rc = cuda_fail(es, "device -> host copy of the rows", __FILE__, __LINE__);
    }
    float ms = 0.f;
    if (rc == MLCC_OK) cudaEventElapsedTime(&ms, ev0, ev1);
    if (rc != MLCC_OK) return rc;
    if (!fin.done) {
        set_last_error("internal: state machine did not finish");
        return MLCC_ERR_CUDA;
    }
    if (out_stats) {
        out_stats->root_iterations = fin.root_iterations;
        out_stats->star_pairs = fin.root_iterations * N;
        out_stats->root_pairs = (fin.root_iterations - fin.root_iterations_noA) * (n_r - 1);
        out_stats->kernel_launches = launches;
        out_stats->total_iterations = fin.total_iterations;
        out_stats->steps = max_steps + 1;
        out_stats->subchains = n_sub;
        out_stats->predictor_order = order;
        out_stats->unconverged_rows = fin.unconverged_rows;
        out_stats->degenerate_roots = fin.degenerate;
        out_stats->solve_ms = ms;
        out_stats->aberth_sum_precision = mode == MODE_F64 ? 64 : 32;
        out_stats->regime = MLCC_REGIME_TILED;
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
