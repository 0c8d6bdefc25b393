// phx_kernels.cu — hand-written sm_100a kernels of the phx hot path.
//
//   k_step8           : a3, fused AdamW step + bf16 copy + packed snapshot (include/phx.h).
//                       Pure HBM streaming: 14 B/element read, 26 B/element written, one pass,
//                       256-bit vectors (LDG.E.256 / STG.E.256, new on sm_100), streaming cache
//                       hints, no shared memory, no tensor cores (no contraction).
//                       MODE bits: kModeF32 = binary32 gradients and no bf16
//                       copy (the paper's precision; 16 B read + 24 B written);
//                       kModeGroups = per-tensor decay groups; kModePublish = the model-param copy also
//                       goes to the peers' parameter buffers (P2P stores, the fused all-gather).
//                       DEV: the derived scalars come from the device-resident step block (graph-capturable form).
//   k_step_prologue   : graph-capturable form: advances the device step counter, derives the AdamW scalars in
//                       binary64 with individually rounded operations and writes the envelope(s).
//   k_sumsq_*         : a1, deterministic fp64 sum of squares + clip coefficient.
//   k_grads_finalize  : SURVEY §8(f4) second half: the gradient producer's epilogue — fp32 main gradients
//                       x scale -> RNE bf16 gradients AND the fp64 sum of squares of the rounded values, one pass.
//   k_regen_bf16      : p16 = RNE_bf16(p).
//   k_restore_bulk    : a6, pulls the replica (a list of 1..3 of its planes) from mapped pinned host memory
//                       with 1-D bulk async copies (TMA, cp.async.bulk + mbarrier) into shared memory, writes
//                       the live planes back with bulk stores and regenerates the bf16 copy from p.
//
// The other flavours tried in round 1 (128-bit vectors, two/four groups per thread, .cs hints, a TMA tile
// pipeline: 5.8-6.4 TB/s against 6.65 for this one) are recorded in profiles/r01_step8_c2_full.md.
//
// Arithmetic contract (include/phx.h a3): every fp32 operation individually rounded —
// __fmul_rn/__fadd_rn/__fsub_rn never fuse into FMA, __fdiv_rn/__fsqrt_rn are IEEE — and the
// file must be compiled WITHOUT --use_fast_math and with the default -ftz=false.
#include "phx_kernels.cuh"

#include <cuda_bf16.h>

namespace phx {

// ------------------------------------------------------------------------------------------
// vector memory helpers.  Streaming hints: loads never allocate in L1 and are marked evict-first in
// L2, stores never allocate in L1 (measured best of the hint combinations, profiles/r01_step8_c2_full.md).
// p/m/v are read then overwritten by the same thread, so the non-coherent (.nc) path is used
// only for the gradients.
// ------------------------------------------------------------------------------------------
struct F8 {
    float x[8];
};

#define PHX_LD256(QUAL)                                                                              \
    asm volatile("ld.global" QUAL ".v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"                          \
                 : "=f"(r.x[0]), "=f"(r.x[1]), "=f"(r.x[2]), "=f"(r.x[3]), "=f"(r.x[4]), "=f"(r.x[5]), \
                   "=f"(r.x[6]), "=f"(r.x[7])                                                         \
                 : "l"(ptr))

__device__ __forceinline__ F8 ld256(const float *ptr)
{
    F8 r;
    PHX_LD256(".L1::no_allocate.L2::evict_first");
    return r;
}
__device__ __forceinline__ void st256(float *ptr, const F8 &r)
{
    asm volatile("st.global.L1::no_allocate.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(ptr), "f"(r.x[0]),
                 "f"(r.x[1]), "f"(r.x[2]), "f"(r.x[3]), "f"(r.x[4]), "f"(r.x[5]), "f"(r.x[6]), "f"(r.x[7])
                 : "memory");
}
// gradients: read-only for the whole kernel -> non-coherent path, never allocate in L1
__device__ __forceinline__ uint4 ldg128_stream(const void *ptr)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(ptr));
    return r;
}
__device__ __forceinline__ F8 ldg256_stream(const float *ptr)
{
    F8 r;
    PHX_LD256(".nc.L1::no_allocate.L2::evict_first");
    return r;
}
__device__ __forceinline__ void st128u(void *ptr, const uint4 &r)
{
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(ptr), "r"(r.x), "r"(r.y), "r"(r.z), "r"(r.w) : "memory");
}

// ------------------------------------------------------------------------------------------
// element arithmetic
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ float bf16lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16hi(uint32_t w) { return __uint_as_float(w & 0xFFFF0000u); }

// two fp32 -> packed bf16x2, round-to-nearest-even (cvt.rn.bf16x2.f32; lo in bits [0,16))
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi)
{
    __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t *>(&h);
}

// One element of the canonical AdamW sequence (include/phx.h a3).  Each intrinsic is one
// IEEE-754 binary32 operation, round-to-nearest-even; none can be contracted into an FMA.
__device__ __forceinline__ void adamw_element(float &p, float &m, float &v, float g, float coef,
                                              const AdamScalars &sc, float decay)
{
    g = __fmul_rn(g, coef);
    const float p1 = __fmul_rn(p, decay);
    const float mn = __fadd_rn(__fmul_rn(sc.beta1, m), __fmul_rn(sc.omb1, g));
    const float vn = __fadd_rn(__fmul_rn(sc.beta2, v), __fmul_rn(sc.omb2, __fmul_rn(g, g)));
    const float d = __fadd_rn(__fdiv_rn(__fsqrt_rn(vn), sc.sbc2), sc.eps);
    p = __fsub_rn(p1, __fmul_rn(sc.ss, __fdiv_rn(mn, d)));
    m = mn;
    v = vn;
}

// ------------------------------------------------------------------------------------------
// 1-D bulk async copy (TMA) + mbarrier helpers (the restore kernel)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    do {  // try_wait suspends the thread in hardware for a bounded time; loop until the phase flips
        asm volatile(
            "{\n"
            ".reg .pred P1;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\n"
            "selp.u32 %0, 1, 0, P1;\n"
            "}\n"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!ok);
}
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gsrc, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_s2g(void *gdst, const void *smem_src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(smem_src)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

// ------------------------------------------------------------------------------------------
// a3: fused step + snapshot, 8 elements per thread-group, 256-bit vectors
// ------------------------------------------------------------------------------------------
constexpr int kStepThreads = 256;

// Decay groups (include/phx.h "decay groups"): cls[e >> kDecayTileShift] says whether the 2048-element
// tile holding e is all-decay (0), all-no-decay (1) or mixed (2); in a mixed tile the flag of element
// e is first_nodecay XOR (number of toggle offsets <= e), found by binary search.  Mixed tiles are
// the few that contain a tensor boundary between a decayed and a no-decay tensor.
__device__ __forceinline__ bool nodecay_at(uint64_t e, const uint64_t *__restrict__ bnd, uint32_t nb, uint32_t first)
{
    uint32_t lo = 0, hi = nb;
    while (lo < hi) {
        const uint32_t mid = (lo + hi) >> 1;
        if (__ldg(bnd + mid) <= e) lo = mid + 1;
        else hi = mid;
    }
    return ((first ^ lo) & 1u) != 0;
}

// Block 0 stores the 256-byte envelope in front of the staging slot (and, §8(f4), a second copy whose
// payload word and hash describe the full rank state) so that the packed snapshot is produced by ONE kernel.
__device__ __forceinline__ void store_headers(const StepArgs &a)
{
    if (blockIdx.x != 0 || threadIdx.x >= 16) return;
    uint4 q = a.hdr.q[threadIdx.x];
    if (a.shdr != nullptr) reinterpret_cast<uint4 *>(a.shdr)[threadIdx.x] = q;
    if (a.shdr_full != nullptr) {
        if (threadIdx.x == 6) q.w = a.full_payload;                 // bytes 108..111
        if (threadIdx.x == 15) {                                    // bytes 240..247
            q.x = (uint32_t)a.full_hash;
            q.y = (uint32_t)(a.full_hash >> 32);
        }
        reinterpret_cast<uint4 *>(a.shdr_full)[threadIdx.x] = q;
    }
}

template <bool SNAP, int MODE, bool DEV>
__global__ void __launch_bounds__(kStepThreads) k_step8(const __grid_constant__ StepArgs a)
{
    constexpr bool GF32 = (MODE & kModeF32) != 0, GROUPS = (MODE & kModeGroups) != 0, PUB = (MODE & kModePublish) != 0;
    const uint64_t gi = (uint64_t)blockIdx.x * kStepThreads + threadIdx.x;
    AdamScalars sc;
    if (DEV) {  // graph-capturable form: k_step_prologue left the scalars (and the envelopes) in device memory
        const float4 s0 = __ldg(reinterpret_cast<const float4 *>(a.dsc));
        const float4 s1 = __ldg(reinterpret_cast<const float4 *>(a.dsc) + 1);
        sc.beta1 = s0.x, sc.beta2 = s0.y, sc.eps = s0.z, sc.decay = s0.w;
        sc.omb1 = s1.x, sc.omb2 = s1.y, sc.ss = s1.z, sc.sbc2 = s1.w;
    } else {
        sc = a.sc;
        store_headers(a);
    }
    if (gi >= (a.n_padded >> 3)) return;
    const float coef = __ldg(a.coef);
    const uint64_t e = gi << 3;

    uint4 G;
    F8 GF;
    if (GF32) GF = ldg256_stream(reinterpret_cast<const float *>(a.g) + e);
    else G = ldg128_stream(reinterpret_cast<const uint16_t *>(a.g) + e);
    F8 P = ld256(a.p + e);
    F8 M = ld256(a.m + e);
    F8 V = ld256(a.v + e);

    float gv[8];
    if (GF32) {
#pragma unroll
        for (int j = 0; j < 8; ++j) gv[j] = GF.x[j];
    } else {
        const uint32_t gw[4] = {G.x, G.y, G.z, G.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            gv[2 * j] = bf16lo(gw[j]);
            gv[2 * j + 1] = bf16hi(gw[j]);
        }
    }
    uint32_t cls = 0;
    if (GROUPS) cls = __ldg(a.decay_cls + (e >> kDecayTileShift));
    if (!GROUPS || cls != 2) {
        const float decay = (GROUPS && cls == 1) ? 1.0f : sc.decay;
#pragma unroll
        for (int j = 0; j < 8; ++j) adamw_element(P.x[j], M.x[j], V.x[j], gv[j], coef, sc, decay);
    } else {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const float decay = nodecay_at(e + j, a.decay_bnd, a.n_bnd, a.first_nodecay) ? 1.0f : sc.decay;
            adamw_element(P.x[j], M.x[j], V.x[j], gv[j], coef, sc, decay);
        }
    }
    st256(a.p + e, P);
    st256(a.m + e, M);
    st256(a.v + e, V);
    if (!GF32) {
        uint4 h;
        h.x = pack_bf16x2(P.x[0], P.x[1]);
        h.y = pack_bf16x2(P.x[2], P.x[3]);
        h.z = pack_bf16x2(P.x[4], P.x[5]);
        h.w = pack_bf16x2(P.x[6], P.x[7]);
        st128u(reinterpret_cast<uint16_t *>(a.p16) + e, h);
        if (PUB)  // all-gather fused into the step: the same 16 bytes go to every peer's buffer (P2P stores)
            for (uint32_t q = 0; q < a.n_pub; ++q) st128u(reinterpret_cast<uint16_t *>(a.pub[q]) + e, h);
    } else if (PUB) {
        for (uint32_t q = 0; q < a.n_pub; ++q) st256(reinterpret_cast<float *>(a.pub[q]) + e, P);
    }
    if (SNAP) {
        st256(a.sp + e, P);
        st256(a.sm + e, M);
        st256(a.sv + e, V);
    }
}

template <int MODE, bool DEV>
static cudaError_t launch8(const StepArgs &a, bool snapshot, cudaStream_t st)
{
    const uint64_t ngroups = a.n_padded >> 3;
    const unsigned grid = (unsigned)((ngroups + kStepThreads - 1) / kStepThreads);
    if (grid == 0) return cudaSuccess;
    if (snapshot) k_step8<true, MODE, DEV><<<grid, kStepThreads, 0, st>>>(a);
    else k_step8<false, MODE, DEV><<<grid, kStepThreads, 0, st>>>(a);
    return cudaGetLastError();
}

// mode: bit set of kMode* (SURVEY §8(f2)/(f3)); dev: the derived scalars come from the device-resident step
// block (a.dsc) instead of the kernel parameters (the graph-capturable form).
cudaError_t launch_step(const StepArgs &a, bool snapshot, uint32_t mode, bool dev, cudaStream_t st)
{
#define PHX_MODE_CASE(M) \
    case M: return dev ? launch8<M, true>(a, snapshot, st) : launch8<M, false>(a, snapshot, st)
    switch (mode) {
        PHX_MODE_CASE(0);
        PHX_MODE_CASE(1);
        PHX_MODE_CASE(2);
        PHX_MODE_CASE(3);
        PHX_MODE_CASE(4);
        PHX_MODE_CASE(5);
        PHX_MODE_CASE(6);
        PHX_MODE_CASE(7);
    default: return cudaErrorInvalidValue;
    }
#undef PHX_MODE_CASE
}

// ------------------------------------------------------------------------------------------
// Graph-capturable form (include/phx.h "graph"): the per-step scalars and the envelope are DERIVED ON THE
// DEVICE from a device-resident step counter, so that a captured step carries no per-step kernel parameter.
// One thread.  Every binary64 operation is an individually rounded intrinsic (__dmul_rn, __dsub_rn,
// __ddiv_rn, __dsqrt_rn) in the same order as the host code of phx_api.cu, so the fp32 results are the same
// bits (tests/test_gpu_graph.py compares them with the oracle for t up to 10^6).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ double pow_sqmul_dev(double b, uint64_t t)  // LSB-first square-and-multiply
{
    double r = 1.0;
    while (t) {
        if (t & 1) r = __dmul_rn(r, b);
        b = __dmul_rn(b, b);
        t >>= 1;
    }
    return r;
}
__device__ __forceinline__ void derive_scalars_dev(float lr, float beta1, float beta2, float eps, float wd, uint64_t t,
                                                   AdamScalars *out)
{
    const double dlr = (double)lr, db1 = (double)beta1, db2 = (double)beta2, dwd = (double)wd;
    out->beta1 = beta1;
    out->beta2 = beta2;
    out->eps = eps;
    out->decay = __double2float_rn(__dsub_rn(1.0, __dmul_rn(dlr, dwd)));
    out->omb1 = __double2float_rn(__dsub_rn(1.0, db1));
    out->omb2 = __double2float_rn(__dsub_rn(1.0, db2));
    out->ss = __double2float_rn(__ddiv_rn(dlr, __dsub_rn(1.0, pow_sqmul_dev(db1, t))));
    out->sbc2 = __double2float_rn(__dsqrt_rn(__dsub_rn(1.0, pow_sqmul_dev(db2, t))));
}
__device__ __forceinline__ uint64_t fnv1a64_dev(const uint8_t *b, int len)
{
    uint64_t h = 0xCBF29CE484222325ull;
    for (int i = 0; i < len; ++i) {
        h ^= b[i];
        h *= 0x100000001B3ull;
    }
    return h;
}

// blk->step += 1; scalars of that step -> blk->sc; envelope of that step (template + step + hash) -> shdr
// and, §8(f4), the full-rank-state flavour -> shdr_full.  expect_slot/expect_depth: the step index the host
// issued this call at, modulo expect_depth = lcm(staging depth, 2) — which fixes both the staging slot and the host
// ping-pong slot baked into the captured nodes; a replay whose device step does not land on it is counted in
// blk->misaligned (phx_graph_end reports it) instead of silently writing the wrong slot.
__global__ void __launch_bounds__(32) k_step_prologue(StepBlock *blk, uint8_t *shdr, uint8_t *shdr_full,
                                                      uint32_t full_payload, uint32_t expect_slot, uint32_t expect_depth)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const uint64_t t = blk->step + 1;
    blk->step = t;
    if (expect_depth != 0 && (uint32_t)(t % expect_depth) != expect_slot) blk->misaligned += 1;
    derive_scalars_dev(blk->lr, blk->beta1, blk->beta2, blk->eps, blk->wd, t, &blk->sc);
    if (shdr == nullptr && shdr_full == nullptr) return;
    // envelope: the template's constant fields + seq_begin = step = seq_end = t + FNV-1a of bytes [0, 240)
    uint8_t *h = blk->hdr_work;
    for (int i = 0; i < 256; ++i) h[i] = blk->hdr_tmpl[i];
    auto put64 = [&](int off, uint64_t v) {
        for (int i = 0; i < 8; ++i) h[off + i] = (uint8_t)(v >> (8 * i));
    };
    auto put32 = [&](int off, uint32_t v) {
        for (int i = 0; i < 4; ++i) h[off + i] = (uint8_t)(v >> (8 * i));
    };
    put64(16, t);   // seq_begin
    put64(24, t);   // step
    put64(248, t);  // seq_end: the slot commits when this header lands
    if (shdr != nullptr) {
        put32(108, 0u);
        put64(240, fnv1a64_dev(h, 240));
        for (int i = 0; i < 16; ++i) reinterpret_cast<uint4 *>(shdr)[i] = reinterpret_cast<const uint4 *>(h)[i];
    }
    if (shdr_full != nullptr) {
        put32(108, full_payload);
        put64(240, fnv1a64_dev(h, 240));
        for (int i = 0; i < 16; ++i) reinterpret_cast<uint4 *>(shdr_full)[i] = reinterpret_cast<const uint4 *>(h)[i];
    }
}

cudaError_t launch_step_prologue(StepBlock *blk, void *shdr, void *shdr_full, uint32_t full_payload, uint32_t expect_slot,
                                 uint32_t expect_depth, cudaStream_t st)
{
    k_step_prologue<<<1, 32, 0, st>>>(blk, static_cast<uint8_t *>(shdr), static_cast<uint8_t *>(shdr_full), full_payload,
                                      expect_slot, expect_depth);
    return cudaGetLastError();
}

// (re)initialise the step block: hyperparameters, the step the live state stands at, the envelope template
__global__ void __launch_bounds__(32) k_step_block_init(StepBlock *blk, float lr, float beta1, float beta2, float eps,
                                                        float wd, uint64_t step, HeaderBlob tmpl)
{
    if (threadIdx.x < 16) reinterpret_cast<uint4 *>(blk->hdr_tmpl)[threadIdx.x] = tmpl.q[threadIdx.x];
    if (threadIdx.x == 0) {
        blk->lr = lr, blk->beta1 = beta1, blk->beta2 = beta2, blk->eps = eps, blk->wd = wd;
        blk->step = step;
        blk->misaligned = 0;
    }
}
cudaError_t launch_step_block_init(StepBlock *blk, float lr, float beta1, float beta2, float eps, float wd, uint64_t step,
                                   const HeaderBlob &tmpl, cudaStream_t st)
{
    k_step_block_init<<<1, 32, 0, st>>>(blk, lr, beta1, beta2, eps, wd, step, tmpl);
    return cudaGetLastError();
}

// test hook (phx_derived_scalars_device): the device derivation for n step indices -> out[5*i] = {decay, omb1, omb2, ss, sbc2}
__global__ void __launch_bounds__(128) k_derive_scalars(float lr, float beta1, float beta2, float wd,
                                                        const uint64_t *__restrict__ steps, uint32_t n, float *__restrict__ out)
{
    const uint32_t i = blockIdx.x * 128 + threadIdx.x;
    if (i >= n) return;
    AdamScalars sc;
    derive_scalars_dev(lr, beta1, beta2, 0.0f, wd, steps[i], &sc);
    out[5 * i + 0] = sc.decay, out[5 * i + 1] = sc.omb1, out[5 * i + 2] = sc.omb2, out[5 * i + 3] = sc.ss, out[5 * i + 4] = sc.sbc2;
}
cudaError_t launch_derive_scalars(float lr, float beta1, float beta2, float wd, const uint64_t *d_steps, uint32_t n,
                                  float *d_out, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    k_derive_scalars<<<(n + 127) / 128, 128, 0, st>>>(lr, beta1, beta2, wd, d_steps, n, d_out);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// a1: sum of squares (fp64, fixed two-stage tree => deterministic run to run) + clip coefficient
// ------------------------------------------------------------------------------------------
// Widening a bf16 to binary64.  The plain way (widen to fp32, cvt.f64.f32) runs on the XU pipe, 16 lanes per
// clock and SM, while the kernel needs ~13 elements per clock and SM to keep HBM busy: with every element
// converted there, ncu shows XU 75 % busy and DRAM only 77 % (profiles/r01_aux_kernels.md).  So the two
// halves of each 32-bit word take different pipes:
//   low half : cvt.f64.f32 (XU);
//   high half: integer re-bias — for a normal bf16 (exponent field e8 != 0, mantissa m7) the double is
//              (e8 + 896) << 52 | m7 << 45, i.e. high word ((w >> 3) & 0x0FFFE000) + 0x38000000, low word 0
//              (sign dropped: only squares are taken); zeros, subnormals, Inf and NaN (e8 = 0 or 255) fall
//              back to the conversion so that they keep their IEEE meaning.
// x*x is exact in binary64 (16 significant bits), so fma(x, x, acc) is ONE rounding of acc + g^2.
// non-zero iff the high half of ANY of the four words has exponent field E = 0 or 255.  (w + 0x00800000) adds one to
// E (carry into the sign bit, nothing below bit 23 moves), so bits 30..24 of the sum — the low 7 bits of its top
// byte — are all zero iff E + 1 is 0 or 1 mod 256.  The four top bytes are gathered into one word (PRMT) and tested
// with the zero-byte trick: 11 integer operations per 8-element group instead of a compare per word.
__device__ __forceinline__ uint32_t any_hi_special(const uint4 &w)
{
    const uint32_t c = 0x00800000u;
    const uint32_t t01 = __byte_perm(w.x + c, w.y + c, 0x0073);   // byte 0 = top byte of x, byte 1 = top byte of y
    const uint32_t t23 = __byte_perm(w.z + c, w.w + c, 0x0073);
    const uint32_t u = __byte_perm(t01, t23, 0x5410) & 0x7F7F7F7Fu;
    return (u - 0x01010101u) & ~u & 0x80808080u;                    // some byte of u is zero
}
__device__ __forceinline__ double widen_hi_int(uint32_t w)
{
    // high word = ((w & 0x7FFF0000) >> 3) + 0x38000000, the shift and the add as ONE multiply-add-high by 2^29
    uint32_t hi;
    asm("mad.hi.u32 %0, %1, 0x20000000, 0x38000000;" : "=r"(hi) : "r"(w & 0x7FFF0000u));
    return __hiloint2double((int)hi, 0);
}
__device__ __forceinline__ void sq_acc4(double &a0, double &a1, const uint4 &w)
{
    const uint32_t ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const double lo = (double)bf16lo(ww[k]);
        a0 = fma(lo, lo, a0);
    }
    // one branch per 8-element group keeps the conversions of the fallback off the XU pipe in the common case
    if (any_hi_special(w) == 0u) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const double hi = widen_hi_int(ww[k]);
            a1 = fma(hi, hi, a1);
        }
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            float f = bf16hi(ww[k]);
            double hi;
            asm volatile("cvt.f64.f32 %0, %1;" : "=d"(hi) : "f"(f));  // volatile: not hoisted out of the branch
            a1 = fma(hi, hi, a1);
        }
    }
}

// The three reduction kernels below share ONE shape (profiles/r02_structure_probe.md: short-lived CTAs stream
// 8-12 % faster than a persistent grid-stride loop on every read:write mix):
//   one-shot CTAs of 256 threads; thread t of CTA b takes the kSumsqK groups (b*kSumsqK + j)*256 + t, j = 0..K-1,
//   of 8 consecutive elements each, issues all its loads at once, accumulates in TWO fixed chains (low halves /
//   even elements, high halves / odd elements, groups in order j), adds the chains, and the CTA reduces
//   (xor-shuffle tree, then the 8 warp sums in order) to partials[b].  k_sumsq_final folds the
//   ceil(ngroups / (256 K)) partials: thread t sums partials[t], partials[t + 1024], ... in order, then a
//   1024-wide tree.  The shape depends on n alone => deterministic run to run, and IDENTICAL between a1 over
//   bf16 gradients and the producer epilogue over the same (rounded) values: the two sums are equal bit for bit.
__device__ __forceinline__ void block_reduce_to_partial(double acc, double *__restrict__ partials)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, o);
    __shared__ double wsum[8];
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = wsum[0];
#pragma unroll
        for (int k = 1; k < 8; ++k) s += wsum[k];
        partials[blockIdx.x] = s;
    }
}

// a1 over bf16 gradients: 128-bit loads (8 gradients each), kSumsqBatchA1 in flight per thread.
__global__ void __launch_bounds__(256) k_sumsq_partial(const uint16_t *__restrict__ g, uint64_t ngroups,
                                                       double *__restrict__ partials)
{
    double acc = 0.0, acc1 = 0.0;
    const uint64_t g0 = (uint64_t)blockIdx.x * (256 * kSumsqK) + threadIdx.x;
#pragma unroll 1
    for (int b = 0; b < kSumsqK; b += kSumsqBatchA1) {
        uint4 w[kSumsqBatchA1];
#pragma unroll
        for (int j = 0; j < kSumsqBatchA1; ++j) {
            const uint64_t gi = g0 + (uint64_t)(b + j) * 256;
            w[j] = gi < ngroups ? ldg128_stream(g + (gi << 3)) : make_uint4(0u, 0u, 0u, 0u);
        }
#pragma unroll
        for (int j = 0; j < kSumsqBatchA1; ++j)
            if (g0 + (uint64_t)(b + j) * 256 < ngroups) sq_acc4(acc, acc1, w[j]);
    }
    block_reduce_to_partial(acc + acc1, partials);
}

// binary32 gradients: the square of a widened fp32 value is exact in fp64 (48 bits),
// so fma(x, x, acc) rounds exactly once, like a separate exact multiply and an add.
__device__ __forceinline__ double sq_acc_f32(double acc, float g)
{
    const double x = (double)g;
    return acc + x * x;
}

__global__ void __launch_bounds__(256) k_sumsq_partial_f32(const float *__restrict__ g, uint64_t ngroups,
                                                           double *__restrict__ partials)
{
    double acc = 0.0, acc1 = 0.0;
    const uint64_t g0 = (uint64_t)blockIdx.x * (256 * kSumsqK) + threadIdx.x;
#pragma unroll 1
    for (int b = 0; b < kSumsqK; b += kSumsqBatchG32) {
        F8 w[kSumsqBatchG32];
#pragma unroll
        for (int j = 0; j < kSumsqBatchG32; ++j) {
            const uint64_t gi = g0 + (uint64_t)(b + j) * 256;
            if (gi < ngroups) w[j] = ldg256_stream(g + (gi << 3));
        }
#pragma unroll
        for (int j = 0; j < kSumsqBatchG32; ++j)
            if (g0 + (uint64_t)(b + j) * 256 < ngroups) {
#pragma unroll
                for (int e = 0; e < 8; e += 2) {
                    acc = sq_acc_f32(acc, w[j].x[e]);
                    acc1 = sq_acc_f32(acc1, w[j].x[e + 1]);
                }
            }
    }
    block_reduce_to_partial(acc + acc1, partials);
}

__global__ void __launch_bounds__(kSumsqMaxBlocks) k_sumsq_final(const double *__restrict__ partials, uint64_t count,
                                                                 float max_norm, double *__restrict__ out_sumsq,
                                                                 float *__restrict__ out_coef)
{
    __shared__ double sh[kSumsqMaxBlocks];
    double a = 0.0;  // 0.0 + x == x: for count <= 1024 this is the plain 1024-wide tree over the partials
#pragma unroll 8
    for (uint64_t i = threadIdx.x; i < count; i += kSumsqMaxBlocks) a += partials[i];
    sh[threadIdx.x] = a;
    __syncthreads();
    for (int o = kSumsqMaxBlocks / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double S = sh[0];
        double c = (double)max_norm / (sqrt(S) + 1e-6);  // IEEE double sqrt and divide
        if (c > 1.0) c = 1.0;
        *out_sumsq = S;
        if (out_coef != nullptr) *out_coef = (float)c;  // cvt.rn.f32.f64
    }
}

uint64_t sumsq_partials_count(uint64_t n_padded)
{
    const uint64_t ngroups = n_padded >> 3, per = 256ull * kSumsqK;
    const uint64_t c = (ngroups + per - 1) / per;
    return c < 1 ? 1 : c;
}

cudaError_t launch_sumsq_clip(const void *g, bool grads_f32, uint64_t n_padded, float max_norm, double *partials,
                              double *out_sumsq, float *out_coef, cudaStream_t st, int *n_launches)
{
    const uint64_t ngroups = n_padded >> 3, nblocks = sumsq_partials_count(n_padded);
    if (nblocks > 0x7FFFFFFFull) return cudaErrorInvalidValue;
    if (grads_f32) k_sumsq_partial_f32<<<(unsigned)nblocks, 256, 0, st>>>(reinterpret_cast<const float *>(g), ngroups, partials);
    else k_sumsq_partial<<<(unsigned)nblocks, 256, 0, st>>>(reinterpret_cast<const uint16_t *>(g), ngroups, partials);
    k_sumsq_final<<<1, kSumsqMaxBlocks, 0, st>>>(partials, nblocks, max_norm, out_sumsq, out_coef);
    if (n_launches) *n_launches = 2;
    return cudaGetLastError();
}

// §8(e) global clip, first half: S_r of this rank's gradient shard -> *out_sumsq (no coefficient)
cudaError_t launch_sumsq(const void *g, bool grads_f32, uint64_t n_padded, double *partials, double *out_sumsq,
                         cudaStream_t st, int *n_launches)
{
    return launch_sumsq_clip(g, grads_f32, n_padded, 0.0f, partials, out_sumsq, nullptr, st, n_launches);
}

// §8(e) global clip, second half: S = sum of `count` per-rank values (same fixed tree) -> coefficient
cudaError_t launch_clip_from_partials(const double *partials, uint32_t count, float max_norm, double *out_sumsq,
                                      float *out_coef, cudaStream_t st)
{
    if (count < 1 || count > (uint32_t)kSumsqMaxBlocks) return cudaErrorInvalidValue;
    k_sumsq_final<<<1, kSumsqMaxBlocks, 0, st>>>(partials, count, max_norm, out_sumsq, out_coef);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// SURVEY §8(f4), second half — the gradient producer's epilogue (reading R34): ONE pass that
// reads the binary32 main gradients (the reduce-scatter output of the ZeRO-2 optimizer),
// writes the optimizer's bf16 gradients  g16 = RNE_bf16(g32 * scale)  and leaves the fp64 per-block sums
// of widen(g16)^2 — the squares of the ROUNDED values, i.e. exactly what a1 would compute from g16 — so
// that the step needs no pass of its own over the gradients (phx_set_clip_partials, count = 1).
// 4 B read + 2 B written per element; the same one-shot shape and tree as a1 => the same sum, bit for bit.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_grads_finalize(const float *__restrict__ g32, float scale, void *__restrict__ g16,
                                                        uint64_t ngroups, double *__restrict__ partials)
{
    double acc = 0.0, acc1 = 0.0;
    const uint64_t g0 = (uint64_t)blockIdx.x * (256 * kSumsqK) + threadIdx.x;
#pragma unroll 1
    for (int b = 0; b < kSumsqK; b += kSumsqBatchF32) {
        F8 w[kSumsqBatchF32];
#pragma unroll
        for (int j = 0; j < kSumsqBatchF32; ++j) {
            const uint64_t gi = g0 + (uint64_t)(b + j) * 256;
            if (gi < ngroups) w[j] = ldg256_stream(g32 + (gi << 3));
        }
#pragma unroll
        for (int j = 0; j < kSumsqBatchF32; ++j) {
            const uint64_t gi = g0 + (uint64_t)(b + j) * 256;
            if (gi < ngroups) {
                const F8 &f = w[j];
                uint4 h;  // cvt.rn.bf16x2.f32 of the individually rounded products
                h.x = pack_bf16x2(__fmul_rn(f.x[0], scale), __fmul_rn(f.x[1], scale));
                h.y = pack_bf16x2(__fmul_rn(f.x[2], scale), __fmul_rn(f.x[3], scale));
                h.z = pack_bf16x2(__fmul_rn(f.x[4], scale), __fmul_rn(f.x[5], scale));
                h.w = pack_bf16x2(__fmul_rn(f.x[6], scale), __fmul_rn(f.x[7], scale));
                st128u(reinterpret_cast<uint16_t *>(g16) + (gi << 3), h);
                sq_acc4(acc, acc1, h);
            }
        }
    }
    block_reduce_to_partial(acc + acc1, partials);
}

cudaError_t launch_grads_finalize(const float *g32, float scale, void *g16, uint64_t n_padded, double *partials,
                                  double *out_sumsq, cudaStream_t st, int *n_launches)
{
    const uint64_t ngroups = n_padded >> 3, nblocks = sumsq_partials_count(n_padded);
    if (nblocks > 0x7FFFFFFFull) return cudaErrorInvalidValue;
    k_grads_finalize<<<(unsigned)nblocks, 256, 0, st>>>(g32, scale, g16, ngroups, partials);
    k_sumsq_final<<<1, kSumsqMaxBlocks, 0, st>>>(partials, nblocks, 0.0f, out_sumsq, nullptr);
    if (n_launches) *n_launches = 2;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// p16 = RNE_bf16(p)
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_regen_bf16(const float *__restrict__ p, void *__restrict__ p16, uint64_t ngroups)
{
    const uint64_t gi = (uint64_t)blockIdx.x * 256 + threadIdx.x;
    if (gi >= ngroups) return;
    const F8 P = ld256(p + (gi << 3));
    uint4 h;
    h.x = pack_bf16x2(P.x[0], P.x[1]);
    h.y = pack_bf16x2(P.x[2], P.x[3]);
    h.z = pack_bf16x2(P.x[4], P.x[5]);
    h.w = pack_bf16x2(P.x[6], P.x[7]);
    st128u(reinterpret_cast<uint16_t *>(p16) + (gi << 3), h);
}

cudaError_t launch_regen_bf16(const float *p, void *p16, uint64_t n_padded, cudaStream_t st)
{
    const uint64_t ngroups = n_padded >> 3;
    if (ngroups == 0) return cudaSuccess;
    k_regen_bf16<<<(unsigned)((ngroups + 255) / 256), 256, 0, st>>>(p, p16, ngroups);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// a6: restore from the mapped pinned host replica with 1-D bulk async copies (TMA).
//   Takes a PLANE LIST (1..3 of p, m, v): all three for the one-phase restore; {p} and then {m, v} (or, full rank
//   state, {p, m, v} behind W) for the two-phase restore of phx_restore_async.
//   Per CTA: kStages shared-memory stages of 3 x kTile fp32 (one tile per plane).  One elected
//   thread arms an mbarrier with the byte count and issues one cp.async.bulk load
//   host -> smem per plane and tile; when they land it issues the cp.async.bulk stores smem -> live
//   planes (no register traffic), while all threads read the tile of plane 0 (p) from smem, convert to
//   bf16 and store the copy (p16 != nullptr).  The host link (PCIe) is the bound: 148 x 2 CTAs keep
//   296 x kStages x 24 KB of reads in flight, but FOUR CTAs already saturate it (profiles/r02c_restore_bulk.md),
//   which is what the second phase runs on so that the recomputed iteration keeps the other SMs.
// ------------------------------------------------------------------------------------------
constexpr int kTile = 2048;  // elements per plane per tile (8 KB)
constexpr int kStages = 4;
constexpr int kRestoreThreads = 256;

__global__ void __launch_bounds__(kRestoreThreads) k_restore_bulk(const __grid_constant__ RestorePlanes pl,
                                                                  void *__restrict__ p16, uint64_t n_padded)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float *tiles = reinterpret_cast<float *>(smem_raw);  // [kStages][3][kTile]
    __shared__ __align__(8) uint64_t full[kStages];

    const int np = pl.n;  // 1..3 planes: {p, m, v}, {p} (parameters first) or {m, v} (two-phase restore)
    const uint64_t ntiles = (n_padded + kTile - 1) / kTile;
    const uint64_t my_first = blockIdx.x;
    const uint64_t stride = gridDim.x;
    const uint64_t my_count = my_first < ntiles ? (ntiles - my_first + stride - 1) / stride : 0;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    auto issue = [&](uint64_t it) {  // thread 0 only
        const int s = (int)(it % kStages);
        const uint64_t t = my_first + it * stride;
        const uint64_t e0 = t * kTile;
        const uint32_t cnt = (uint32_t)((n_padded - e0) < (uint64_t)kTile ? (n_padded - e0) : kTile);
        const uint32_t bytes = cnt * 4u;
        float *dst = tiles + (size_t)s * 3 * kTile;
        mbar_expect_tx(&full[s], (uint32_t)np * bytes);
        for (int k = 0; k < np; ++k) bulk_g2s(dst + k * kTile, pl.src[k] + e0, bytes, &full[s]);
    };

    if (threadIdx.x == 0)
        for (uint64_t it = 0; it < my_count && it < (uint64_t)kStages; ++it) issue(it);

    for (uint64_t it = 0; it < my_count; ++it) {
        const int s = (int)(it % kStages);
        const uint32_t parity = (uint32_t)((it / kStages) & 1);
        const uint64_t t = my_first + it * stride;
        const uint64_t e0 = t * kTile;
        const uint32_t cnt = (uint32_t)((n_padded - e0) < (uint64_t)kTile ? (n_padded - e0) : kTile);
        float *tp = tiles + (size_t)s * 3 * kTile;
        mbar_wait(&full[s], parity);
        if (threadIdx.x == 0) {
            for (int k = 0; k < np; ++k) bulk_s2g(pl.dst[k] + e0, tp + k * kTile, cnt * 4u);
            bulk_commit();
        }
        // bf16 copy of plane 0 (p): 8 elements per thread, conflict-free 128-bit shared loads
        const uint32_t e = threadIdx.x * 8;
        if (p16 != nullptr && e < cnt) {
            const float4 a = *reinterpret_cast<const float4 *>(tp + e);
            const float4 b = *reinterpret_cast<const float4 *>(tp + e + 4);
            uint4 h;
            h.x = pack_bf16x2(a.x, a.y);
            h.y = pack_bf16x2(a.z, a.w);
            h.z = pack_bf16x2(b.x, b.y);
            h.w = pack_bf16x2(b.z, b.w);
            st128u(reinterpret_cast<uint16_t *>(p16) + e0 + e, h);
        }
        __syncthreads();  // everyone is done reading stage s
        if (threadIdx.x == 0) {
            bulk_wait_read0();  // the bulk stores have finished reading stage s
            if (it + kStages < my_count) issue(it + kStages);
        }
    }
    if (threadIdx.x == 0) bulk_wait_all0();  // stores globally complete before the CTA exits
}

cudaError_t launch_restore_bulk(const RestorePlanes &pl, void *p16, uint64_t n_padded, int max_ctas, cudaStream_t st)
{
    if (n_padded == 0) return cudaSuccess;
    if (pl.n < 1 || pl.n > 3) return cudaErrorInvalidValue;
    const size_t smem = (size_t)kStages * 3 * kTile * sizeof(float);  // 96 KB
    // function attributes are per DEVICE: set it on every launch (a cheap host-side call) rather than behind a
    // process-wide flag, which left the second GPU of a one-process-many-GPUs caller without the opt-in
    cudaError_t e = cudaFuncSetAttribute(k_restore_bulk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const uint64_t ntiles = (n_padded + kTile - 1) / kTile;
    uint64_t grid = max_ctas > 0 ? (uint64_t)max_ctas : 1;
    if (grid > ntiles) grid = ntiles;
    k_restore_bulk<<<(unsigned)grid, kRestoreThreads, smem, st>>>(pl, p16, n_padded);
    return cudaGetLastError();
}

}  // namespace phx
