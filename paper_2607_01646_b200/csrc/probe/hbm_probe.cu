// hbm_probe.cu — BENCH-ONLY diagnostic (see phx_probe.h); a library of its own, not linked into libphx.so.
#include "phx_probe.h"

#include <cuda_runtime.h>

namespace {

constexpr int kStepThreads = 256;
constexpr int kProbeMaxPlanes = 8;

struct F8 {
    float x[8];
};
__device__ __forceinline__ F8 ld256(const float *ptr)
{
    F8 r;
    asm volatile("ld.global.L1::no_allocate.L2::evict_first.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(r.x[0]), "=f"(r.x[1]), "=f"(r.x[2]), "=f"(r.x[3]), "=f"(r.x[4]), "=f"(r.x[5]), "=f"(r.x[6]),
                   "=f"(r.x[7])
                 : "l"(ptr));
    return r;
}
__device__ __forceinline__ void st256(float *ptr, const F8 &r)
{
    asm volatile("st.global.L1::no_allocate.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(ptr), "f"(r.x[0]),
                 "f"(r.x[1]), "f"(r.x[2]), "f"(r.x[3]), "f"(r.x[4]), "f"(r.x[5]), "f"(r.x[6]), "f"(r.x[7])
                 : "memory");
}

// ------------------------------------------------------------------------------------------
// Diagnostic: the HBM ceiling of a read:write mix.  One pass over n_read + n_write disjoint planes
// with the fused step's access pattern (one 256-bit vector per thread and plane, the same cache
// hints, 256-thread CTAs) and NO arithmetic beyond what keeps the loads alive.  bench.py reports the
// fused kernel against the ceiling of its own mix (3 fp32 planes read, 6 written) next to the
// driver-measured copy peak.  RT/WT >= 0: compile-time plane counts (few registers, full occupancy,
// used for the mixes bench.py reports); -1: run-time counts (any mix up to 8 + 8 planes).
// ------------------------------------------------------------------------------------------
template <int RT, int WT>
__device__ __forceinline__ void probe_group(float *__restrict__ base, uint64_t plane_elems, uint64_t gi, uint32_t n_read_rt,
                                            uint32_t n_write_rt)
{
    constexpr int RMAX = RT >= 0 ? (RT > 0 ? RT : 1) : kProbeMaxPlanes;
    constexpr int WMAX = WT >= 0 ? (WT > 0 ? WT : 1) : kProbeMaxPlanes;
    const int n_read = RT >= 0 ? RT : (int)n_read_rt, n_write = WT >= 0 ? WT : (int)n_write_rt;
    const uint64_t e = gi << 3;
    F8 acc;
#pragma unroll
    for (int j = 0; j < 8; ++j) acc.x[j] = (float)(uint32_t)gi;
    F8 r[RMAX];
#pragma unroll
    for (int i = 0; i < RMAX; ++i)
        if (i < n_read) r[i] = ld256(base + (uint64_t)i * plane_elems + e);
#pragma unroll
    for (int i = 0; i < RMAX; ++i)
        if (i < n_read) {
#pragma unroll
            for (int j = 0; j < 8; ++j) acc.x[j] = __fadd_rn(acc.x[j], r[i].x[j]);
        }
#pragma unroll
    for (int i = 0; i < WMAX; ++i)
        if (i < n_write) st256(base + (uint64_t)(n_read + i) * plane_elems + e, acc);
    if (n_write == 0) {  // keep the loads alive: a store that never happens
        float t = 0.f;
#pragma unroll
        for (int j = 0; j < 8; ++j) t += acc.x[j];
        if (t == -123.456f) base[e] = t;
    }
}

// one-shot structure (the fused step's): one 8-element group per thread, ceil(ngroups/256) short-lived CTAs
template <int RT, int WT>
__global__ void __launch_bounds__(kStepThreads) k_hbm_probe(float *__restrict__ base, uint64_t plane_elems, uint64_t ngroups,
                                                            uint32_t n_read_rt, uint32_t n_write_rt)
{
    const uint64_t gi = (uint64_t)blockIdx.x * kStepThreads + threadIdx.x;
    if (gi < ngroups) probe_group<RT, WT>(base, plane_elems, gi, n_read_rt, n_write_rt);
}

// persistent structure: 148 x ctas_per_sm CTAs walking the groups with a grid stride (the alternative design for a
// streaming kernel; measured 8-12 % SLOWER than the one-shot structure on every mix, profiles/r02_structure_probe.md)
template <int RT, int WT>
__global__ void __launch_bounds__(kStepThreads) k_hbm_probe_persistent(float *__restrict__ base, uint64_t plane_elems,
                                                                       uint64_t ngroups, uint32_t n_read_rt, uint32_t n_write_rt)
{
    const uint64_t stride = (uint64_t)gridDim.x * kStepThreads;
    for (uint64_t gi = (uint64_t)blockIdx.x * kStepThreads + threadIdx.x; gi < ngroups; gi += stride)
        probe_group<RT, WT>(base, plane_elems, gi, n_read_rt, n_write_rt);
}

cudaError_t launch_hbm_probe(void *d_buf, uint64_t plane_bytes, uint32_t n_read, uint32_t n_write, uint32_t persistent_grid,
                             cudaStream_t st)
{
    if (n_read > (uint32_t)kProbeMaxPlanes || n_write > (uint32_t)kProbeMaxPlanes || n_read + n_write == 0)
        return cudaErrorInvalidValue;
    const uint64_t plane_elems = plane_bytes / 4, ngroups = plane_elems >> 3;
    if (ngroups == 0) return cudaSuccess;
    const unsigned grid = (unsigned)((ngroups + kStepThreads - 1) / kStepThreads);
    float *b = static_cast<float *>(d_buf);
#define PHX_PROBE(R, W)                                                                                          \
    do {                                                                                                         \
        if (persistent_grid)                                                                                     \
            k_hbm_probe_persistent<R, W><<<persistent_grid, kStepThreads, 0, st>>>(b, plane_elems, ngroups, n_read, n_write); \
        else                                                                                                     \
            k_hbm_probe<R, W><<<grid, kStepThreads, 0, st>>>(b, plane_elems, ngroups, n_read, n_write);          \
    } while (0)
    switch (n_read * 16 + n_write) {
    case 4 * 16 + 0: PHX_PROBE(4, 0); break;
    case 0 * 16 + 4: PHX_PROBE(0, 4); break;
    case 1 * 16 + 1: PHX_PROBE(1, 1); break;
    case 3 * 16 + 6: PHX_PROBE(3, 6); break;
    case 3 * 16 + 3: PHX_PROBE(3, 3); break;
    case 2 * 16 + 1: PHX_PROBE(2, 1); break;
    default: PHX_PROBE(-1, -1); break;
    }
#undef PHX_PROBE
    return cudaGetLastError();
}

}  // namespace

static int probe_impl(void *d_buf, uint64_t plane_bytes, uint32_t n_read, uint32_t n_write, uint32_t persistent_grid, void *stream)
{
    if (!d_buf || plane_bytes == 0 || (plane_bytes & 255u) || n_read > (uint32_t)kProbeMaxPlanes ||
        n_write > (uint32_t)kProbeMaxPlanes || n_read + n_write == 0)
        return -1;
    if (reinterpret_cast<uintptr_t>(d_buf) & 255u) return -2;
    if (launch_hbm_probe(d_buf, plane_bytes, n_read, n_write, persistent_grid, static_cast<cudaStream_t>(stream)) != cudaSuccess) {
        (void)cudaGetLastError();
        return -9;
    }
    return 0;
}

extern "C" int phx_hbm_probe_async(void *d_buf, uint64_t plane_bytes, uint32_t n_read, uint32_t n_write, void *stream)
{
    return probe_impl(d_buf, plane_bytes, n_read, n_write, 0u, stream);
}

extern "C" int phx_hbm_probe_persistent_async(void *d_buf, uint64_t plane_bytes, uint32_t n_read, uint32_t n_write,
                                              uint32_t grid, void *stream)
{
    if (grid == 0) return -1;
    return probe_impl(d_buf, plane_bytes, n_read, n_write, grid, stream);
}
