// chain.cu — the small-field regime of the critical-curve solver: one CTA owns one sub-chain and runs all of its
// rows and all of their Aberth–Ehrlich iterations by itself (SURVEY.md §7 "kernel regimes": n_r = 20 ... a few
// thousand roots per phase; PAPER.md:211 "if the GPU threads are not already saturated", :213 sub-chains).
//
// Same mathematics as aberth.cu (Eq. 15 / 17 / 19):
//   Delta_k = F / (F' + F (2 S1 - A)),  z_k <- z_k - Delta_k,  frozen once |Delta_k| < tol,
// Jacobi (every step of an iteration is taken from the same iterate), seeds z_i +/- 1 for the cold
// centre row, polynomial predictor through the chain's last rows for the others (R18),
// confirming iterations without the Aberth sum (R27), caustic point from the same sums (Eq. 12).
//
// Why a second regime: for N <~ 10^3 stars one iteration of all rows in flight is a few microseconds of arithmetic,
// and the tiled path (aberth.cu) spends five dependent launches on it.  Here nothing leaves the SM between the
// first seed and the last row of a sub-chain:
//   * stars, the current iterate of the two rows being solved (the sub-chain grows from its centre row towards
//     both ends, one row each way per step: PAPER.md:211), the steps and the lists of unfrozen roots live in
//     shared memory; the only global traffic is the finished rows (16 B per root and per caustic point) and the
//     predictor's reads of the chain's last rows (L2 hits: this CTA wrote them);
//   * an iteration is: pair loops -> __syncthreads -> apply + ordered compaction -> __syncthreads;
//   * the unfrozen entries are worked off in passes that keep every thread busy: two adjacent entries per thread
//     (each shared-memory read of a source serves both) while there are that many, one per thread, then T lanes of
//     a warp per entry (T = 2 .. 32), combined by shuffles in a fixed order: two runs give the same bits.
// All arithmetic is FP64; the reciprocal of the Aberth sum is the 20-bit seed (R19), that of the star sums full.
#include "star_sums.cuh"
#include "predictor.cuh"

#include <math.h>
#include <algorithm>
#include <vector>

namespace mlcc {
namespace {

#ifndef MLCC_CHAIN_MIN_CTAS
#define MLCC_CHAIN_MIN_CTAS 1
#endif
#ifndef MLCC_CHAIN_MAX_THREADS
#define MLCC_CHAIN_MAX_THREADS 512
#endif
constexpr int CR = 2;                 // list entries per thread
constexpr double TINY = 1e-300;       // |d|^2 + TINY: the pair of a root with itself contributes exactly 0


struct ChainCounters {
    unsigned long long root_iterations;       // unfrozen roots updated, summed over iterations, rows and sub-chains
    unsigned long long root_iterations_noA;   // ... of which without the Aberth sum
    int max_iterations;                       // longest sequence of iterations run by one CTA (the critical path)
    int unconverged_rows;
    int degenerate;
    int pad;
};

struct ChainParams {
    const double2 *stars;
    const double *masses;
    int N;
    int n_r;
    double gamma, omk, tol2, skip_below2;
    int max_iter, max_iter_cold, order;
    const double2 *rot;          // [num_phi] (1-kappa_s) e^{-i phi_j}
    const double2 *init_roots;   // [n_r] or null
    double2 *roots;              // [num_phi][n_r]
    double2 *caustics;           // [num_phi][n_r] or null
    int *out_iters, *out_unconverged;
    const long long *sub_first, *sub_centre, *sub_end;
    ChainCounters *counters;
};

__device__ __forceinline__ void pair_root(double zx, double zy, double2 r, double &ax, double &ay)
{
    const double dx = zx - r.x;
    const double dy = r.y - zy;
    const double r2 = fma(dy, dy, fma(dx, dx, TINY));
    const double inv = rcp_seed(r2);
    ax = fma(dx, inv, ax);
    ay = fma(dy, inv, ay);
}

// sum over the CTA of a 64-bit value, the same result in every thread (s_buf: 33 entries)
__device__ __forceinline__ unsigned long long block_sum(unsigned long long v, unsigned long long *s_buf)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = (blockDim.x + 31) >> 5;
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if (lane == 0) s_buf[warp] = v;
    __syncthreads();
    unsigned long long t = 0;
    for (int w = 0; w < nwarps; ++w) t += s_buf[w];
    return t;
}

// 0 frozen, 1 iterated next with the Aberth sum, 2 iterated next without it (the same predicate as aberth.cu)
__device__ __forceinline__ int step_kind(double d2, double tol2, double skip2)
{
    if (d2 < tol2) return 0;
    return d2 < skip2 ? 2 : 1;
}

// One pass of the pair loops over the list entries [base, base + RR blockDim.x / T): lane group g = tid / T takes the
// RR adjacent entries base + g RR + r, lane sub = tid % T the sources sub, sub + T, ... of each; the T shares are
// combined by shuffles in a fixed order and lane 0 of the group takes the Aberth step (into s_delta, by entry) and
// writes the caustic point.  Entries below n_large get the Aberth sum, the others the Newton step of F (R27).
template <bool CAUS, int RR, bool EQM>
__device__ __forceinline__ void chain_pass(const ChainParams &p, double m0, int base, int T, int n_act, int n_large,
                                           const int *__restrict__ list, const double2 *__restrict__ s_xy,
                                           const double *__restrict__ s_m, const double2 *__restrict__ s_z,
                                           double2 *__restrict__ s_delta, const long long *row_s)
{
    const int N = p.N, n_r = p.n_r, tid = threadIdx.x;
    const int sub = tid & (T - 1), grp = tid / T;
    int e[RR], set[RR];
    bool valid[RR], large[RR];
    double zx[RR], zy[RR];
    StarAcc acc[RR];
    double ax[RR], ay[RR];
#pragma unroll
    for (int r = 0; r < RR; ++r) {
        const int pos = base + grp * RR + r;
        valid[r] = pos < n_act;
        large[r] = pos < n_large;
        e[r] = valid[r] ? list[pos] : list[0];
        set[r] = e[r] >= n_r ? 1 : 0;
        const double2 z = s_z[e[r]];
        zx[r] = z.x;
        zy[r] = z.y;
        acc[r] = StarAcc{0, 0, 0, 0, 0, 0, 0, 0};
        ax[r] = ay[r] = 0.0;
    }
    if (valid[0]) {
        // star sums (S1 only where the Aberth sum is used)
        if (large[0]) {
#pragma unroll (RR == 1 ? 4 : 2)
            for (int j = sub; j < N; j += T) {
                const double2 s = s_xy[j];
                const double m = EQM ? 0.0 : s_m[j];
#pragma unroll
                for (int r = 0; r < RR; ++r) {
                    if (EQM) pair_star_eq<CAUS, true>(zx[r], zy[r], s, acc[r]);
                    else pair_star<CAUS, true>(zx[r], zy[r], s, m, acc[r]);
                }
            }
        } else {
#pragma unroll (RR == 1 ? 4 : 2)
            for (int j = sub; j < N; j += T) {
                const double2 s = s_xy[j];
                const double m = EQM ? 0.0 : s_m[j];
#pragma unroll
                for (int r = 0; r < RR; ++r) {
                    if (EQM) pair_star_eq<CAUS, false>(zx[r], zy[r], s, acc[r]);
                    else pair_star<CAUS, false>(zx[r], zy[r], s, m, acc[r]);
                }
            }
        }
        if (EQM) {
#pragma unroll
            for (int r = 0; r < RR; ++r) {
                if (large[0]) star_sums_scale<CAUS, true>(acc[r], m0);
                else star_sums_scale<CAUS, false>(acc[r], m0);
            }
        }
        // Aberth sum over the current iterate of the entry's own row
        if (RR == 2 && large[0] && large[RR - 1] && valid[RR - 1] && set[0] == set[RR - 1]) {
            const double2 *src = s_z + set[0] * n_r;
#pragma unroll 2
            for (int j = sub; j < n_r; j += T) {
                const double2 s = src[j];
#pragma unroll
                for (int r = 0; r < RR; ++r) pair_root(zx[r], zy[r], s, ax[r], ay[r]);
            }
        } else {
#pragma unroll
            for (int r = 0; r < RR; ++r) {
                if (!(valid[r] && large[r])) continue;
                const double2 *src = s_z + set[r] * n_r;
#pragma unroll 4
                for (int j = sub; j < n_r; j += T) pair_root(zx[r], zy[r], src[j], ax[r], ay[r]);
            }
        }
    }
    // ---- combine the T shares (fixed order), one Aberth step per entry ----
#pragma unroll
    for (int r = 0; r < RR; ++r) {
        double v[CAUS ? 8 : 6] = {2.0 * acc[r].s1x - ax[r], 2.0 * acc[r].s1y - ay[r], acc[r].s2x, acc[r].s2h,
                                  acc[r].s3x, acc[r].s3y};
        if (CAUS) { v[6] = acc[r].smx; v[7] = acc[r].smy; }
        for (int o = T >> 1; o > 0; o >>= 1)
#pragma unroll
            for (int q = 0; q < (CAUS ? 8 : 6); ++q) v[q] += __shfl_xor_sync(0xffffffffu, v[q], o);
        if (valid[r] && sub == 0) {
            const long long row = row_s[set[r]];
            const int k = e[r] - set[r] * n_r;
            const double2 rot = p.rot[row];
            // without the Aberth sum the step is the Newton step of F (R27): t = 2 S1 - A left out
            const double tx = large[r] ? v[0] : 0.0, ty = large[r] ? v[1] : 0.0;
            const double s2x = v[2], s2y = 2.0 * v[3], s3x = v[4], s3y = v[5];
            const double fx = p.gamma + s2x - rot.x, fy = s2y - rot.y;   // F
            const double gx = -2.0 * s3x, gy = -2.0 * s3y;               // F'
            const double dnx = gx + (fx * tx - fy * ty);                 // F' + F (2 S1 - A)
            const double dny = gy + (fx * ty + fy * tx);
            const double dn2 = dnx * dnx + dny * dny;
            double2 d;
            d.x = (fx * dnx + fy * dny) / dn2;
            d.y = (fy * dnx - fx * dny) / dn2;
            s_delta[e[r]] = d;
            if (CAUS) {
                // caustic point of z - Delta from the sums at z (second order in Delta; exact to rounding once the
                // root freezes): Sm(z - D) = Sm + D S2 + D^2 S3
                const double d2x = d.x * d.x - d.y * d.y, d2y = 2.0 * d.x * d.y;
                const double mx = v[6] + (d.x * s2x - d.y * s2y) + (d2x * s3x - d2y * s3y);
                const double my = v[7] + (d.x * s2y + d.y * s2x) + (d2x * s3y + d2y * s3x);
                const double nx = zx[r] - d.x, ny = zy[r] - d.y;
                double2 w;
                w.x = fma(p.omk + p.gamma, nx, -mx);
                w.y = fma(p.omk - p.gamma, ny, my);
                p.caustics[row * n_r + k] = w;
            }
        }
    }
}

template <bool CAUS>
__global__ void __launch_bounds__(MLCC_CHAIN_MAX_THREADS, MLCC_CHAIN_MIN_CTAS) k_chain(ChainParams p)
{
    extern __shared__ __align__(16) unsigned char s_raw[];
    __shared__ unsigned long long s_buf[33];
    __shared__ int s_warp[33];
    const int N = p.N, n_r = p.n_r, NT = blockDim.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nwarps = (NT + 31) >> 5;
    double2 *s_xy = reinterpret_cast<double2 *>(s_raw);                 // [N]
    double2 *s_z = s_xy + N;                                            // [2][n_r] current iterate of the two rows
    double2 *s_delta = s_z + 2 * n_r;                                   // [2 n_r] steps of this iteration, by entry
    double *s_m = reinterpret_cast<double *>(s_delta + 2 * n_r);        // [N]
    int *s_list = reinterpret_cast<int *>(s_m + N + (N & 1));           // [2][2 n_r] unfrozen entries, ping-pong

    const int c = blockIdx.x;
    const long long first = p.sub_first[c], centre = p.sub_centre[c], end = p.sub_end[c];
    const int max_step = (int)max(centre - first, end - 1 - centre);
    for (int i = tid; i < N; i += NT) {
        s_xy[i] = p.stars[i];
        s_m[i] = p.masses[i];
    }
    __syncthreads();
    // a field of equal masses takes the lighter pair body (star_sums.cuh); decided here, the same in every thread
    const double m0 = s_m[0];
    int same = 1;
    for (int i = tid; i < N; i += NT) same &= (s_m[i] == m0);
    const bool eqm = __syncthreads_and(same) != 0;
    unsigned long long n_rootit = 0, n_rootit_noA = 0;   // thread 0's tallies
    int n_iter_total = 0, n_unconv_rows = 0, n_degenerate = 0;

    for (int step = 0; step <= max_step; ++step) {
        // rows of this step: set 0 = downward (the centre row itself at step 0), set 1 = upward
        const long long row_s[2] = {centre - step, centre + step};
        const bool has_s[2] = {row_s[0] >= first, step > 0 && row_s[1] < end};
        int cur = 0;
        // ---- seeds, identity lists ----
        int n_act = 0;
        for (int set = 0; set < 2; ++set) {
            if (!has_s[set]) continue;
            const long long row = row_s[set];
            const int dir = set == 0 ? -1 : +1;
            int order = 0;
            if (step > 0) {
                const long long room = (dir > 0) ? (row - first) : (end - 1 - row);
                const long long avail = min((long long)(2 * step - 1), room);
                order = (int)min((long long)p.order, avail - 1);
            }
            for (int k = tid; k < n_r; k += NT) {
                double2 z;
                if (step == 0) {
                    if (p.init_roots) {
                        z = p.init_roots[k];
                    } else {   // z_i + 1, z_i - 1
                        const int i = (k < N) ? k : k - N;
                        z = s_xy[i];
                        z.x += (k < N) ? 1.0 : -1.0;
                    }
                } else {
                    double2 v[PRED_MAX_ORDER + 1];
#pragma unroll
                    for (int q = 0; q <= PRED_MAX_ORDER; ++q)
                        v[q] = q <= order ? __ldcg(&p.roots[(row - (long long)dir * (q + 1)) * n_r + k])
                                          : make_double2(0.0, 0.0);
                    z = predict_adaptive(v, order);
                }
                s_z[set * n_r + k] = z;
                s_list[n_act + k] = set * n_r + k;
            }
            n_act += n_r;
        }
        int n_small = 0;                      // entries [n_act - n_small, n_act) of the list skip the Aberth sum
        int rem[2] = {has_s[0] ? n_r : 0, has_s[1] ? n_r : 0};
        int iters_row[2] = {0, 0};
        int iter = 0;
        const int cap = step == 0 ? p.max_iter_cold : p.max_iter;
        __syncthreads();

        while (n_act > 0 && iter < cap) {
            const int *list = s_list + cur * 2 * n_r;
            int *next = s_list + (cur ^ 1) * 2 * n_r;
            const int n_large = n_act - n_small;
            // ---- pair loops.  A pass gives every lane group RR adjacent list entries and splits the sources of an
            // entry over the T lanes of its group (the schedule of the passes is below). ----
            // The entries that keep the Aberth sum and those that do not cost different amounts per entry, so the two
            // groups get passes of their own: inside a pass every thread then does the same work.
            for (int seg = 0; seg < 2; ++seg) {
                const int seg_end = seg == 0 ? n_large : n_act;
                for (int base = seg == 0 ? 0 : n_large; base < seg_end;) {
                    const int left = seg_end - base;
                    // Passes that keep every thread busy: two entries per thread while at least 2 NT are left, one entry
                    // per thread while at least NT are left, then the remainder over T lanes per entry with T the
                    // largest power of two that still gives every thread a share (a remainder above NT / 2 takes two
                    // such passes).  A pass in which some warps have nothing to do makes them wait at the barrier for
                    // its whole length (ncu: 23 % of the warp samples of cfg2 sat there with the earlier schedule).
                    int rr = 1, T = 1;
                    if (left >= 2 * NT) {
                        rr = 2;
                    } else if (left >= NT) {
                    } else {
                        T = 2;
                        while (T < 32 && left * (2 * T) <= NT) T <<= 1;
                    }
                    if (eqm) {
                        if (rr == 2) chain_pass<CAUS, 2, true>(p, m0, base, T, seg_end, n_large, list, s_xy, s_m, s_z, s_delta, row_s);
                        else chain_pass<CAUS, 1, true>(p, m0, base, T, seg_end, n_large, list, s_xy, s_m, s_z, s_delta, row_s);
                    } else {
                        if (rr == 2) chain_pass<CAUS, 2, false>(p, m0, base, T, seg_end, n_large, list, s_xy, s_m, s_z, s_delta, row_s);
                        else chain_pass<CAUS, 1, false>(p, m0, base, T, seg_end, n_large, list, s_xy, s_m, s_z, s_delta, row_s);
                    }
                    base += rr * NT / T;
                }
            }
            __syncthreads();
            // ---- apply the steps, freeze, compact in order: survivors with the Aberth sum first, then the others ----
            // pass 1: how many of each kind, and how many survivors per row
            // four 16-bit tallies in one word (2 n_r < 65536 by the shared-memory limit):
            // survivors with the Aberth sum | survivors of row 0 << 16 | of row 1 << 32 | non-finite steps << 48
            unsigned long long cnt = 0;
            for (int pos = tid; pos < n_act; pos += NT) {
                const int ee = list[pos];
                const double2 d = s_delta[ee];
                const double d2 = d.x * d.x + d.y * d.y;
                if (d2 <= 1.79769313486231570e308) {
                    const int kind = step_kind(d2, p.tol2, p.skip_below2);
                    if (kind == 1) cnt += 1ull;
                    if (kind != 0) cnt += (ee >= n_r) ? (1ull << 32) : (1ull << 16);
                } else {
                    cnt += 1ull << 48;   // NaN / Inf: the root is frozen where it is and reported
                }
            }
            const unsigned long long tot = block_sum(cnt, s_buf);
            const int next_large = (int)(tot & 0xffffull);
            const int rem0 = (int)((tot >> 16) & 0xffffull), rem1 = (int)((tot >> 32) & 0xffffull);
            const int bad_total = (int)(tot >> 48);
            // pass 2: ordered write
            int base_l = 0, base_s = next_large;
            for (int c0 = 0; c0 < n_act; c0 += NT * CR) {
                int ks[CR], kind[CR];
                int pc = 0;
#pragma unroll
                for (int i = 0; i < CR; ++i) {
                    const int pos = c0 + tid * CR + i;
                    kind[i] = 0;
                    ks[i] = 0;
                    if (pos < n_act) {
                        const int ee = list[pos];
                        const double2 d = s_delta[ee];
                        const double d2 = d.x * d.x + d.y * d.y;
                        if (d2 <= 1.79769313486231570e308) {
                            double2 z = s_z[ee];
                            z.x -= d.x;
                            z.y -= d.y;
                            s_z[ee] = z;
                            kind[i] = step_kind(d2, p.tol2, p.skip_below2);
                        }
                        ks[i] = ee;
                        pc += kind[i] == 1 ? 1 : (kind[i] == 2 ? (1 << 16) : 0);
                    }
                }
                int incl = pc;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int n = __shfl_up_sync(0xffffffffu, incl, o);
                    if (lane >= o) incl += n;
                }
                if (lane == 31) s_warp[warp] = incl;
                __syncthreads();
                if (warp == 0) {
                    const int w = lane < nwarps ? s_warp[lane] : 0;
                    int wi = w;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int n = __shfl_up_sync(0xffffffffu, wi, o);
                        if (lane >= o) wi += n;
                    }
                    s_warp[lane] = wi - w;
                    if (lane == 31) s_warp[32] = wi;
                }
                __syncthreads();
                const int excl = s_warp[warp] + incl - pc;
                int off_l = base_l + (excl & 0xffff), off_s = base_s + (excl >> 16);
#pragma unroll
                for (int i = 0; i < CR; ++i) {
                    if (kind[i] == 1) next[off_l++] = ks[i];
                    else if (kind[i] == 2) next[off_s++] = ks[i];
                }
                const int tot2 = s_warp[32];
                base_l += tot2 & 0xffff;
                base_s += tot2 >> 16;
                __syncthreads();
            }
            // ---- bookkeeping (the same values in every thread) ----
            iter += 1;
            if (rem[0] > 0) iters_row[0] = iter;
            if (rem[1] > 0) iters_row[1] = iter;
            n_rootit += (unsigned long long)n_act;
            n_rootit_noA += (unsigned long long)n_small;
            n_degenerate += bad_total;
            rem[0] = rem0;
            rem[1] = rem1;
            n_act = base_s;
            n_small = base_s - next_large;
            cur ^= 1;
        }
        n_iter_total += iter;
        // ---- the rows are final: write them, with their diagnostics ----
        for (int set = 0; set < 2; ++set) {
            if (!has_s[set]) continue;
            const long long row = row_s[set];
            for (int k = tid; k < n_r; k += NT) p.roots[row * n_r + k] = s_z[set * n_r + k];
            if (tid == 0) {
                if (p.out_iters) p.out_iters[row] = iters_row[set];
                if (p.out_unconverged) p.out_unconverged[row] = rem[set];
            }
            if (rem[set] > 0) ++n_unconv_rows;
        }
        __syncthreads();   // the rows are read back by the next step's predictor; s_list / s_z are rewritten
    }
    if (tid == 0) {
        atomicAdd(&p.counters->root_iterations, n_rootit);
        atomicAdd(&p.counters->root_iterations_noA, n_rootit_noA);
        atomicMax(&p.counters->max_iterations, n_iter_total);
        if (n_unconv_rows) atomicAdd(&p.counters->unconverged_rows, n_unconv_rows);
        if (n_degenerate) atomicAdd(&p.counters->degenerate, n_degenerate);
    }
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
size_t chain_smem_bytes(int64_t N, int64_t n_r)
{
    return (size_t)N * 16 + (size_t)(N + (N & 1)) * 8 + (size_t)n_r * (2 * 16 + 2 * 16 + 4 * 4);
}

int chain_threads(int64_t n_r)
{
    // two rows of n_r roots per step, R entries per thread, four lanes per root wanted when that is small
    long long nt = (2 * n_r * 4 + CR - 1) / CR;
    nt = (nt + 31) / 32 * 32;
    if (nt < 32) nt = 32;
    if (nt > MLCC_CHAIN_MAX_THREADS) nt = MLCC_CHAIN_MAX_THREADS;
    return (int)nt;
}

// How many chain CTAs are resident at once (0: this field does not fit the regime).
int chain_capacity(int64_t N, int64_t n_r, bool caus)
{
    const size_t smem = chain_smem_bytes(N, n_r);
    int dev = 0, max_optin = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (smem + 1024 > (size_t)max_optin) return 0;
    auto fn = caus ? k_chain<true> : k_chain<false>;
    if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, chain_threads(n_r), smem) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    return per_sm * device_sm_count();
}

struct ChainRun {
    unsigned long long root_iterations, root_iterations_noA;
    int max_iterations, unconverged_rows, degenerate;
};

// Runs the whole solve: one launch, one CTA per sub-chain.  `counters` [1] device scratch (zeroed here).
int chain_launch(const double *star_xy, const double *masses, int64_t N, int64_t n_r, double gamma, double omk,
                 double tol, double skip_below, int max_iter, int max_iter_cold, int order, const void *d_rot,
                 const double *init_roots, double *roots, double *caustics, int *out_iters, int *out_unconverged,
                 int n_sub, const long long *d_first, const long long *d_centre, const long long *d_end,
                 void *d_counters, cudaStream_t stream)
{
    ChainParams p{};
    p.stars = reinterpret_cast<const double2 *>(star_xy);
    p.masses = masses;
    p.N = (int)N;
    p.n_r = (int)n_r;
    p.gamma = gamma;
    p.omk = omk;
    p.tol2 = tol * tol;
    p.skip_below2 = skip_below > 0.0 ? skip_below * skip_below : 0.0;
    p.max_iter = max_iter;
    p.max_iter_cold = max_iter_cold;
    p.order = order;
    p.rot = static_cast<const double2 *>(d_rot);
    p.init_roots = reinterpret_cast<const double2 *>(init_roots);
    p.roots = reinterpret_cast<double2 *>(roots);
    p.caustics = reinterpret_cast<double2 *>(caustics);
    p.out_iters = out_iters;
    p.out_unconverged = out_unconverged;
    p.sub_first = d_first;
    p.sub_centre = d_centre;
    p.sub_end = d_end;
    p.counters = static_cast<ChainCounters *>(d_counters);
    MLCC_CUDA(cudaMemsetAsync(d_counters, 0, sizeof(ChainCounters), stream));
    const size_t smem = chain_smem_bytes(N, n_r);
    auto fn = caustics ? k_chain<true> : k_chain<false>;
    MLCC_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    fn<<<n_sub, chain_threads(n_r), smem, stream>>>(p);
    MLCC_CUDA(cudaGetLastError());
    return MLCC_OK;
}

size_t chain_counters_bytes() { return sizeof(ChainCounters); }

void chain_read_counters(const void *h_counters, ChainRun *out)
{
    const ChainCounters *c = static_cast<const ChainCounters *>(h_counters);
    out->root_iterations = c->root_iterations;
    out->root_iterations_noA = c->root_iterations_noA;
    out->max_iterations = c->max_iterations;
    out->unconverged_rows = c->unconverged_rows;
    out->degenerate = c->degenerate;
}

}  // namespace mlcc
