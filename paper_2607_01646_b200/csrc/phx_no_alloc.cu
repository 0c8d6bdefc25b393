// phx_no_alloc.cu — phx_grad_sumsq_no_alloc (include/phx.h): the sum of squared gradients of a rank's gradient
// shard (the S_r of SURVEY.md §8(e); the a1 pass) for callers that must not allocate device memory.
//
// Why it exists.  phx_grad_sumsq_async needs a BOUND handle, and phx_shard_bind obtains the reduction scratch (one
// fp64 partial per 16384 gradients) with cudaMalloc.  Three kinds of caller of this library cannot afford that call:
//   * a trainer whose framework allocator has already taken the whole HBM (a job sized to the brim of the 180 GB):
//     a driver allocation made behind the framework's back fails, or succeeds and pushes the framework into an
//     out-of-memory error a few iterations later;
//   * anything on the iteration's critical path: cudaMalloc/cudaFree synchronise the device, so one such call from
//     a monitoring thread stalls the snapshot flush and the forward/backward kernels it is meant to hide behind —
//     exactly the checkpoint stall the path is built to avoid;
//   * the fault-handling side (a health check that wants a rank's gradient norm right after a failure was
//     signalled; the recovery procedure of PAPER.md:171): it runs when the allocator's state is the least
//     trustworthy and should not depend on memory being obtainable at all.
// For them the scratch is the file-scope array below: part of the library image, resident on every GPU that loads
// libphx.so from the moment the module is loaded until the process exits (512 KiB per GPU, never freed).
//
// The kernels are the library's own k_sumsq_partial / k_sumsq_partial_f32 / k_sumsq_final with the same launch shape
// (phx::launch_sumsq), so the result has the same bits as phx_grad_sumsq_async on the same gradients.
//
// What a user must know (repeated beside the declaration in phx.h):
//   * One array per GPU, shared by every call and every thread.  Two calls whose kernels may run at the same time
//     on one GPU (different streams with no ordering between them) race on it and both results are garbage.
//     Calls on one stream, or ordered by events, are safe.
//   * The array keeps whatever the previous call left in it.  Nothing has to be cleared: a call with n elements
//     overwrites partials [0, ceil(n / 16384)) in its first kernel and its second kernel reads exactly that range,
//     so stale entries of an earlier, larger call are never read.
//   * The first call on each device looks the array's device address up (cudaGetSymbolAddress; this also makes the
//     driver load the module on that device) under a process-wide mutex.  Make that first call outside any stream
//     capture.  Later calls only enqueue two kernels.
#include "../../include/phx.h"
#include "phx_kernels.cuh"

#include <mutex>

namespace {

constexpr uint64_t kElemsPerPartial = 8ull * 256ull * phx::kSumsqK;  // one reduction CTA: 256 threads x K groups of 8
constexpr uint64_t kMaxPartials = PHX_NO_ALLOC_MAX_ELEMS / kElemsPerPartial;
static_assert(kElemsPerPartial == 16384, "phx.h states one partial per 16384 elements");
static_assert(PHX_NO_ALLOC_MAX_ELEMS % kElemsPerPartial == 0, "the maximum must be a whole number of partials");
static_assert(kMaxPartials * sizeof(double) == 512 * 1024, "phx.h and README.md state 512 KiB per GPU");

// The scratch.  In HOST code this name is only a handle for the runtime's symbol table — not a device address; a
// kernel handed `g_sumsq_scratch` itself would fault (or, on a system where the GPU can reach host memory, scribble
// over host memory).  Host code below therefore uses the address cudaGetSymbolAddress returns, and nothing else.
static __device__ __align__(256) double g_sumsq_scratch[kMaxPartials];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
double *g_scratch_addr[kMaxDevices] = {};  // per device ordinal: device address of g_sumsq_scratch, once looked up

// Once per device, with that device current (it is: we read the ordinal from cudaGetDevice just before).
int scratch_for_current_device(double **out, int *cuda_error)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        if (cuda_error) *cuda_error = (int)e;
        return PHX_ERR_CUDA;
    }
    if (dev < 0 || dev >= kMaxDevices) return PHX_ERR_UNSUPPORTED_DEVICE;
    std::lock_guard<std::mutex> lock(g_mu);
    if (g_scratch_addr[dev] == nullptr) {
        int major = 0;
        e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e == cudaSuccess && major != 10) return PHX_ERR_UNSUPPORTED_DEVICE;  // sm_100a image only, no fallback
        double *p = nullptr;
        if (e == cudaSuccess) e = cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_sumsq_scratch);
        if (e != cudaSuccess || p == nullptr) {
            if (cuda_error) *cuda_error = (int)e;
            (void)cudaGetLastError();
            return PHX_ERR_CUDA;
        }
        g_scratch_addr[dev] = p;
    }
    *out = g_scratch_addr[dev];
    return PHX_OK;
}

}  // namespace

extern "C" int phx_grad_sumsq_no_alloc(const void *d_grads, int grads_fp32, uint64_t n_elems, double *d_out,
                                       void *stream, int *cuda_error)
{
    if (cuda_error) *cuda_error = 0;
    if (!d_grads || !d_out || n_elems == 0 || (n_elems & 7u) || (grads_fp32 != 0 && grads_fp32 != 1))
        return PHX_ERR_INVALID_ARG;
    if (n_elems > PHX_NO_ALLOC_MAX_ELEMS) return PHX_ERR_TOO_LARGE;
    if ((reinterpret_cast<uintptr_t>(d_grads) & 255u) || (reinterpret_cast<uintptr_t>(d_out) & 7u))
        return PHX_ERR_ALIGNMENT;
    double *scratch = nullptr;
    const int rc = scratch_for_current_device(&scratch, cuda_error);
    if (rc != PHX_OK) return rc;
    const cudaError_t e = phx::launch_sumsq(d_grads, grads_fp32 != 0, n_elems, scratch, d_out,
                                            static_cast<cudaStream_t>(stream), nullptr);
    if (e != cudaSuccess) {
        if (cuda_error) *cuda_error = (int)e;
        return PHX_ERR_CUDA;
    }
    return PHX_OK;
}
