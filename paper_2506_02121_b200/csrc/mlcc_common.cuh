// mlcc_common.cuh — shared host/device helpers of libmlcc (product path; not used by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>
#include <stdint.h>
#include <stdio.h>
#include <string>

#include "../../include/mlcc.h"

namespace mlcc {

// ---- error plumbing -------------------------------------------------------------------------
void set_last_error(const std::string &msg);
int cuda_fail(cudaError_t e, const char *what, const char *file, int line);

#define MLCC_CUDA(call)                                                              \
    do {                                                                             \
        cudaError_t e__ = (call);                                                    \
        if (e__ != cudaSuccess) return ::mlcc::cuda_fail(e__, #call, __FILE__, __LINE__); \
    } while (0)

inline int invalid(const char *msg)
{
    set_last_error(std::string("invalid argument: ") + msg);
    return MLCC_ERR_INVALID_ARG;
}

// The stream-ordered allocator gives freed memory back to the driver at every synchronisation unless told
// otherwise, and every call here would then pay for fresh device allocations (hundreds of ms for the GB-sized
// scratch of the matcher): the first library call on a device raises the release threshold of that device's
// DEFAULT memory pool to "keep everything".  This is a process-wide setting of the CUDA runtime: other users of
// cudaMallocAsync on the same device (PyTorch's default caching allocator is not one) keep their freed blocks
// cached too until cudaMemPoolTrimTo is called.  Documented in include/mlcc.h.
void keep_pool_memory();

// Stream-ordered workspace that frees itself (cudaFreeAsync) when it goes out of scope.
struct Workspace {
    static constexpr int CAP = 64;
    cudaStream_t stream;
    void *ptrs[CAP];
    int n = 0;
    explicit Workspace(cudaStream_t s) : stream(s) { keep_pool_memory(); }
    Workspace(const Workspace &) = delete;
    Workspace &operator=(const Workspace &) = delete;
    ~Workspace()
    {
        for (int i = n - 1; i >= 0; --i) cudaFreeAsync(ptrs[i], stream);
    }
    template <typename T>
    cudaError_t alloc(T **out, size_t count)
    {
        *out = nullptr;
        if (n >= CAP) return cudaErrorMemoryAllocation;   // never hand out a block that would not be freed
        void *p = nullptr;
        cudaError_t e = cudaMallocAsync(&p, count * sizeof(T) > 0 ? count * sizeof(T) : 16, stream);
        if (e != cudaSuccess) return e;
        ptrs[n++] = p;
        *out = static_cast<T *>(p);
        return cudaSuccess;
    }
};

// Small owners, so that every early return releases what the call created.
struct Event {
    cudaEvent_t e = nullptr;
    Event() = default;
    Event(const Event &) = delete;
    Event &operator=(const Event &) = delete;
    ~Event() { if (e) cudaEventDestroy(e); }
    cudaError_t create(unsigned flags = cudaEventDefault) { return cudaEventCreateWithFlags(&e, flags); }
    operator cudaEvent_t() const { return e; }
};
struct OwnedStream {
    cudaStream_t s = nullptr;
    OwnedStream() = default;
    OwnedStream(const OwnedStream &) = delete;
    OwnedStream &operator=(const OwnedStream &) = delete;
    ~OwnedStream() { if (s) { cudaStreamSynchronize(s); cudaStreamDestroy(s); } }
    cudaError_t create() { return cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking); }
    operator cudaStream_t() const { return s; }
};
// Pinned host block kept per host thread (cudaMallocHost / cudaFreeHost per call cost 80-120 ms every few calls
// on the bench box); freed when the thread ends (at process exit the runtime may already be gone: the error of
// that late cudaFreeHost is ignored).
struct PinnedBlock {
    void *p = nullptr;
    size_t bytes = 0;
    PinnedBlock() = default;
    PinnedBlock(const PinnedBlock &) = delete;
    PinnedBlock &operator=(const PinnedBlock &) = delete;
    ~PinnedBlock() { if (p) { cudaFreeHost(p); cudaGetLastError(); } }
    cudaError_t reserve(size_t n)
    {
        if (n <= bytes) return cudaSuccess;
        if (p) { cudaFreeHost(p); p = nullptr; bytes = 0; }
        cudaError_t e = cudaMallocHost(&p, n);
        if (e == cudaSuccess) bytes = n;
        return e;
    }
};

int device_sm_count();

// NVTX range on the calling host thread (SURVEY.md §5 "Tracing"): every C-ABI entry point opens one named after the
// call; the solver adds one per phase of its work (set-up, every enqueued chunk of iterations, the final read-back)
// and a mark whenever a poll of the device state shows that further steps of the continuation have finished.  The
// iterations themselves run from a device-side state machine, so per-step ranges exist only as those marks.
// Header-only NVTX 3: no tool attached = a no-op call.
struct NvtxRange {
    explicit NvtxRange(const char *name) { nvtxRangePushA(name); }
    NvtxRange(const NvtxRange &) = delete;
    NvtxRange &operator=(const NvtxRange &) = delete;
    ~NvtxRange() { nvtxRangePop(); }
};

// ---- device arithmetic ------------------------------------------------------------------------
#ifdef __CUDACC__

// MUFU.RCP64H seed of 1/x: the instruction reads only the high word of x and writes only the high
// word of the result (sign, exponent, top 20 mantissa bits; relative error <= 2^-19.9, measured).
// The low word is taken from x itself instead of being zeroed: that moves the seed by < 2^-20
// relative, which is inside its own error, and saves one move per reciprocal.
__device__ __forceinline__ double rcp_seed(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return __hiloint2double(__double2hiint(y), __double2loint(x));
}

// 1/x to ~2 ulp for normal positive x: one cubically convergent step from the seed,
// y1 = y0 (1 + e + e^2), e = 1 - x y0  (error e^3 < 2^-56 before rounding).  No slow path.
__device__ __forceinline__ double rcp_full(double x)
{
    double y = rcp_seed(x);
    double e = fma(-x, y, 1.0);
    double t = fma(e, e, e);
    return fma(y, t, y);
}

#endif  // __CUDACC__

}  // namespace mlcc
