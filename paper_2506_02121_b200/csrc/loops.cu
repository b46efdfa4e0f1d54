// loops.cu — chains and closed loops (fn. 5 at :217).
//
// "Every one of the initial n_r roots begins and ends a 'chain' of values from 0 to 2 pi ... sometimes 2 or more
// chains are needed to fully create a closed critical curve"; "the start of one chain is the end of another, with
// chains joining together until closed loops are formed".  Input is the successor table of mlcc_link_rows.
//
//   chain k starts in column k of row 0;  chain_col[s+1][k] = next[s][chain_col[s][k]];
//   chain_end[k] = next[S-1][chain_col[S-1][k]] is the column of row 0 at which chain k arrives after the whole
//   turn of phi; the loops are the cycles of k -> chain_end[k].
//
// Tracing one chain is S dependent loads.  The S row permutations are composed in blocks of ~sqrt(S) rows instead:
// (1) every (block, column) thread follows its column through the rows of the block -> the block's permutation;
// (2) one thread per chain composes the ~sqrt(S) block permutations -> the chain's column at every block start and
// its end; (3) every (block, chain) thread follows its chain through the block again and writes chain_col.
// ~3 sqrt(S) dependent loads per thread, sqrt(S) n threads in flight, all stores coalesced over k.
// The cycles are labelled by pointer jumping: after r rounds label[k] = min of k, sigma(k), ..., sigma^(2^r - 1)(k)
// and jump[k] = sigma^(2^r)(k); 2^r >= n covers any cycle.  Integer work only: results are exact and reproducible.
#include "mlcc_common.cuh"

namespace mlcc {
namespace {

constexpr int BLOCK = 256;

__global__ void __launch_bounds__(BLOCK) k_block_perm(const int *__restrict__ next, long long S, int n, int rows_per_block,
                                                      int *__restrict__ perm)
{
    const int k = blockIdx.x * BLOCK + threadIdx.x;
    const int b = blockIdx.y;
    if (k >= n) return;
    const long long s0 = (long long)b * rows_per_block;
    const long long s1 = s0 + rows_per_block < S ? s0 + rows_per_block : S;
    int c = k;
    for (long long s = s0; s < s1 && c >= 0; ++s) {
        c = next[s * n + c];
        if ((unsigned)c >= (unsigned)n) c = -1;
    }
    perm[(long long)b * n + k] = c;
}

__global__ void __launch_bounds__(BLOCK) k_block_start(const int *__restrict__ perm, int B, int n, int *__restrict__ start,
                                                       int *__restrict__ chain_end)
{
    const int k = blockIdx.x * BLOCK + threadIdx.x;
    if (k >= n) return;
    int c = k;
    for (int b = 0; b < B; ++b) {
        start[(long long)b * n + k] = c;
        if (c >= 0) c = perm[(long long)b * n + c];
    }
    chain_end[k] = c;
}

__global__ void __launch_bounds__(BLOCK) k_block_write(const int *__restrict__ next, long long S, int n, int rows_per_block,
                                                       const int *__restrict__ start, int *__restrict__ chain_col)
{
    const int k = blockIdx.x * BLOCK + threadIdx.x;
    const int b = blockIdx.y;
    if (k >= n) return;
    const long long s0 = (long long)b * rows_per_block;
    const long long s1 = s0 + rows_per_block < S ? s0 + rows_per_block : S;
    int c = start[(long long)b * n + k];
    for (long long s = s0; s < s1; ++s) {
        chain_col[s * n + k] = c;
        if (c >= 0) {
            c = next[s * n + c];
            if ((unsigned)c >= (unsigned)n) c = -1;
        }
    }
}

__global__ void __launch_bounds__(BLOCK) k_loop_init(const int *__restrict__ chain_end, int n, int *__restrict__ label,
                                                     int *__restrict__ jump, int *__restrict__ on_cycle, int *num_loops)
{
    const int k = blockIdx.x * BLOCK + threadIdx.x;
    if (k == 0) *num_loops = 0;
    if (k >= n) return;
    const int e = chain_end[k];
    label[k] = e < 0 ? -1 : k;
    jump[k] = e;
    on_cycle[k] = 0;
}

__global__ void __launch_bounds__(BLOCK) k_loop_round(const int *__restrict__ label_in, const int *__restrict__ jump_in, int n,
                                                      int *__restrict__ label_out, int *__restrict__ jump_out)
{
    const int k = blockIdx.x * BLOCK + threadIdx.x;
    if (k >= n) return;
    const int l = label_in[k], j = jump_in[k];
    int lo = -1, jo = -1;
    if (l >= 0 && j >= 0) {
        const int lj = label_in[j];
        if (lj >= 0) {
            lo = l < lj ? l : lj;
            jo = jump_in[j];
        }
    }
    label_out[k] = lo;
    jump_out[k] = jo;
}

// sigma^(2^r) maps everything onto the cycles once 2^r >= n: its image is the set of chains that lie on a cycle
__global__ void __launch_bounds__(BLOCK) k_loop_mark(const int *__restrict__ jump, int n, int *__restrict__ on_cycle)
{
    const int k = blockIdx.x * BLOCK + threadIdx.x;
    if (k >= n) return;
    const int j = jump[k];
    if (j >= 0) on_cycle[j] = 1;
}

__global__ void __launch_bounds__(BLOCK) k_loop_final(const int *__restrict__ label, const int *__restrict__ on_cycle, int n,
                                                      int *__restrict__ loop_id, int *num_loops)
{
    const int k = blockIdx.x * BLOCK + threadIdx.x;
    int id = -1;
    if (k < n && on_cycle[k]) id = label[k];
    if (k < n) loop_id[k] = id;
    const int is_root = (k < n && id == k) ? 1 : 0;
    const int total = __syncthreads_count(is_root);
    if (threadIdx.x == 0 && total) atomicAdd(num_loops, total);
}

__global__ void __launch_bounds__(BLOCK) k_order_by_chain(const double2 *__restrict__ points, const int *__restrict__ chain_col,
                                                          long long total, int n, double2 *__restrict__ out)
{
    const double nan = __longlong_as_double(0x7ff8000000000000ll);
    for (long long e = (long long)blockIdx.x * BLOCK + threadIdx.x; e < total; e += (long long)gridDim.x * BLOCK) {
        const long long s = e / n;
        const int c = chain_col[e];
        out[e] = ((unsigned)c < (unsigned)n) ? points[s * n + c] : make_double2(nan, nan);
    }
}

}  // namespace

int closed_loops_impl(const int32_t *next, int64_t S, int64_t n, int32_t *out_chain_col, int32_t *out_chain_end,
                      int32_t *out_loop_id, int32_t *out_num_loops, cudaStream_t stream)
{
    if (!next || !out_chain_end || !out_loop_id || !out_num_loops) return invalid("null pointer");
    if (S < 1 || n < 1 || n > (1 << 30) || S > (1ll << 40)) return invalid("S or n out of range");
    int rows_per_block = 1;
    while ((long long)rows_per_block * rows_per_block < S) ++rows_per_block;       // ceil(sqrt(S))
    const int B = (int)((S + rows_per_block - 1) / rows_per_block);
    if (B > 65535) return invalid("S too large");
    Workspace ws(stream);
    int *perm = nullptr, *start = nullptr, *buf = nullptr;
    cudaError_t e = ws.alloc(&perm, (size_t)B * n);
    if (e == cudaSuccess) e = ws.alloc(&start, (size_t)B * n);
    if (e == cudaSuccess) e = ws.alloc(&buf, (size_t)5 * n);
    if (e == cudaErrorMemoryAllocation) {
        cudaGetLastError();
        set_last_error("workspace allocation failed");
        return MLCC_ERR_NOMEM;
    }
    MLCC_CUDA(e);
    const unsigned gx = (unsigned)((n + BLOCK - 1) / BLOCK);
    k_block_perm<<<dim3(gx, B), BLOCK, 0, stream>>>(next, (long long)S, (int)n, rows_per_block, perm);
    k_block_start<<<gx, BLOCK, 0, stream>>>(perm, B, (int)n, start, out_chain_end);
    if (out_chain_col)
        k_block_write<<<dim3(gx, B), BLOCK, 0, stream>>>(next, (long long)S, (int)n, rows_per_block, start, out_chain_col);
    int *label[2] = {buf, buf + n}, *jump[2] = {buf + 2 * n, buf + 3 * n}, *on_cycle = buf + 4 * n;
    k_loop_init<<<gx, BLOCK, 0, stream>>>(out_chain_end, (int)n, label[0], jump[0], on_cycle, out_num_loops);
    int cur = 0;
    for (long long span = 1; span < n; span *= 2) {
        k_loop_round<<<gx, BLOCK, 0, stream>>>(label[cur], jump[cur], (int)n, label[cur ^ 1], jump[cur ^ 1]);
        cur ^= 1;
    }
    k_loop_mark<<<gx, BLOCK, 0, stream>>>(jump[cur], (int)n, on_cycle);
    k_loop_final<<<gx, BLOCK, 0, stream>>>(label[cur], on_cycle, (int)n, out_loop_id, out_num_loops);
    MLCC_CUDA(cudaGetLastError());
    return MLCC_OK;
}

int order_by_chain_impl(const double *points, const int32_t *chain_col, int64_t S, int64_t n, double *out,
                        cudaStream_t stream)
{
    if (S == 0) return MLCC_OK;
    if (!points || !chain_col || !out) return invalid("null pointer");
    if (S < 1 || n < 1 || n > (1 << 30)) return invalid("S or n out of range");
    if (points == out) return invalid("points and out must not alias");
    const long long total = (long long)S * n;
    long long blocks = (total + BLOCK - 1) / BLOCK;
    const long long cap = 16ll * device_sm_count();       // grid-stride: whole waves of resident CTAs
    if (blocks > cap) blocks = cap;
    k_order_by_chain<<<(unsigned)blocks, BLOCK, 0, stream>>>(reinterpret_cast<const double2 *>(points), chain_col, total,
                                                            (int)n, reinterpret_cast<double2 *>(out));
    MLCC_CUDA(cudaGetLastError());
    return MLCC_OK;
}

}  // namespace mlcc
