// phx_kernels.cuh — internal launch interface between the C-ABI layer (phx_api.cu) and the
// sm_100a kernels (phx_kernels.cu).  Not part of the public boundary (include/phx.h is).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace phx {

// Derived AdamW scalars, computed on the host in double and rounded once (include/phx.h, a3).
struct AdamScalars {
    float beta1, beta2, eps, decay, omb1, omb2, ss, sbc2;
};

// 256-byte envelope passed by value as a kernel parameter; block 0 stores it in front of the
// staging slot so that the packed snapshot (header ‖ p ‖ m ‖ v) is produced by ONE kernel.
struct alignas(16) HeaderBlob {
    uint4 q[16];
};

enum { kMaxPublish = 15 };

struct StepArgs {
    float *p, *m, *v;            // live planes, n_padded each
    const void *g;               // bf16 grads (float grads under kModeF32)
    void *p16;                   // bf16 param copy (unused under kModeF32)
    float *sp, *sm, *sv;         // staging planes of the slot being written (null if !snapshot)
    void *shdr;                  // where block 0 stores the 256-B header (null: no header)
    // §8(f4): second copy of the header for the full-rank-state local slot — same bytes except the
    // payload word (byte 108) and the header hash (byte 240); null: not written
    void *shdr_full;
    uint32_t full_payload;
    uint64_t full_hash;
    const float *coef;           // device scalar: clip coefficient (1.0f when clipping is off)
    uint64_t n_padded;           // multiple of 64
    // decay groups (kModeGroups): class per 2048-element tile, toggle offsets, flag before the first toggle
    const uint8_t *decay_cls;
    const uint64_t *decay_bnd;
    uint32_t n_bnd, first_nodecay;
    // publication (kModePublish): the model-param copy of every element also goes to pub[0..n_pub), the
    // rank's slice inside other DP ranks' parameter buffers (peer HBM over NVLink), already offset
    void *pub[kMaxPublish];
    uint32_t n_pub;
    AdamScalars sc;
    HeaderBlob hdr;
};

enum { kNumStepVariants = 12 };
// SURVEY §8(f2) modes of the fused step (default flavour only): binary32 gradients without a bf16
// copy (the paper's precision) and per-tensor decay groups.
// §8(f3): kModePublish fuses the parameter all-gather into the step (P2P stores into the peers' buffers).
enum { kModeF32 = 1, kModeGroups = 2, kModePublish = 4 };
enum { kDecayTileShift = 11 };  // decay_cls granularity: 2048 elements

// a3.  variant selects the kernel flavour (see phx_kernels.cu); snapshot=false drops the staging stores.
cudaError_t launch_step(const StepArgs &a, bool snapshot, uint32_t variant, uint32_t mode, cudaStream_t st);

// a1.  partials: >= kSumsqMaxBlocks doubles of device scratch; out_sumsq/out_coef device scalars.
enum { kSumsqMaxBlocks = 1024 };
cudaError_t launch_sumsq_clip(const void *g, bool grads_f32, uint64_t n_padded, float max_norm, double *partials,
                              double *out_sumsq, float *out_coef, cudaStream_t st, int *n_launches);

// §8(e) global clip: a1 split around the caller's exchange of per-rank sums (include/phx.h).
cudaError_t launch_sumsq(const void *g, bool grads_f32, uint64_t n_padded, double *partials, double *out_sumsq,
                         cudaStream_t st, int *n_launches);
cudaError_t launch_clip_from_partials(const double *partials, uint32_t count, float max_norm, double *out_sumsq,
                                      float *out_coef, cudaStream_t st);

// p16 = RNE_bf16(p)
cudaError_t launch_regen_bf16(const float *p, void *p16, uint64_t n_padded, cudaStream_t st);

// a6, bulk-kernel mode: src_payload = device-visible address of the host slot's payload (p ‖ m ‖ v);
// p16 == nullptr skips the bf16 regeneration (kModeF32 shards have no bf16 copy).
cudaError_t launch_restore_bulk(const void *src_payload, float *p, float *m, float *v, void *p16,
                                uint64_t n_padded, int sm_count, cudaStream_t st);

// Diagnostic: streaming pass over n_read + n_write planes of plane_bytes each inside d_buf, no arithmetic.
enum { kProbeMaxPlanes = 8 };
cudaError_t launch_hbm_probe(void *d_buf, uint64_t plane_bytes, uint32_t n_read, uint32_t n_write, cudaStream_t st);

}  // namespace phx
