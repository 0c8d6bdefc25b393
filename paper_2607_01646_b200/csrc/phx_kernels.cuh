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
    // graph-capturable form: where k_step_prologue left the scalars of the step (null: use sc and hdr above)
    const AdamScalars *dsc;
    HeaderBlob hdr;
};

// Device-resident step block of the graph-capturable form (include/phx.h "graph"): the hyperparameters, the
// step counter the live state stands at, the scalars k_step_prologue derived for the step in flight, the
// envelope template.  Lives in the handle's device scratch.
struct alignas(16) StepBlock {
    AdamScalars sc;            // must stay first (16-byte aligned vector loads in k_step8<.., DEV>)
    float lr, beta1, beta2, eps, wd;
    uint32_t misaligned;       // replays whose device step did not land on the staging slot baked at capture
    uint64_t step;
    alignas(16) uint8_t hdr_tmpl[256];
    alignas(16) uint8_t hdr_work[256];
};

// SURVEY §8(f2) modes of the fused step (default flavour only): binary32 gradients without a bf16
// copy (the paper's precision) and per-tensor decay groups.
// §8(f3): kModePublish fuses the parameter all-gather into the step (P2P stores into the peers' buffers).
enum { kModeF32 = 1, kModeGroups = 2, kModePublish = 4 };
enum { kDecayTileShift = 11 };  // decay_cls granularity: 2048 elements

// a3.  snapshot=false drops the staging stores; mode = kMode* bits; dev = scalars from a.dsc.
cudaError_t launch_step(const StepArgs &a, bool snapshot, uint32_t mode, bool dev, cudaStream_t st);
// graph-capturable form: ++blk->step, scalars -> blk->sc, envelopes -> shdr / shdr_full (either may be null)
cudaError_t launch_step_prologue(StepBlock *blk, void *shdr, void *shdr_full, uint32_t full_payload, uint32_t expect_slot,
                                 uint32_t expect_depth, cudaStream_t st);
cudaError_t launch_step_block_init(StepBlock *blk, float lr, float beta1, float beta2, float eps, float wd, uint64_t step,
                                   const HeaderBlob &tmpl, cudaStream_t st);
cudaError_t launch_derive_scalars(float lr, float beta1, float beta2, float wd, const uint64_t *d_steps, uint32_t n,
                                  float *d_out, cudaStream_t st);

// a1.  partials: >= sumsq_partials_count(n_padded) doubles of device scratch; out_sumsq/out_coef device scalars.
enum { kSumsqMaxBlocks = 1024 };
#ifndef PHX_SUMSQ_K
#define PHX_SUMSQ_K 8
#endif
#ifndef PHX_SUMSQ_BATCH_A1
#define PHX_SUMSQ_BATCH_A1 8
#endif
#ifndef PHX_SUMSQ_BATCH_F32
#define PHX_SUMSQ_BATCH_F32 8
#endif
// kSumsqK: 8-element groups per thread of the short-lived reduction CTAs (part of the tree's shape);
// kSumsqBatch*: how many of them a thread has in flight at once (loads issued together) — not part of the shape
enum { kSumsqK = PHX_SUMSQ_K, kSumsqBatchA1 = PHX_SUMSQ_BATCH_A1, kSumsqBatchF32 = PHX_SUMSQ_BATCH_F32, kSumsqBatchG32 = 4 };
static_assert(kSumsqK % kSumsqBatchA1 == 0 && kSumsqK % kSumsqBatchF32 == 0, "batches must tile the per-thread groups");
uint64_t sumsq_partials_count(uint64_t n_padded);
cudaError_t launch_sumsq_clip(const void *g, bool grads_f32, uint64_t n_padded, float max_norm, double *partials,
                              double *out_sumsq, float *out_coef, cudaStream_t st, int *n_launches);

// §8(e) global clip: a1 split around the caller's exchange of per-rank sums (include/phx.h).
cudaError_t launch_sumsq(const void *g, bool grads_f32, uint64_t n_padded, double *partials, double *out_sumsq,
                         cudaStream_t st, int *n_launches);
cudaError_t launch_clip_from_partials(const double *partials, uint32_t count, float max_norm, double *out_sumsq,
                                      float *out_coef, cudaStream_t st);

// §8(f4) second half: g16 = RNE_bf16(g32 * scale) and the sum of squares of the rounded values, one pass
cudaError_t launch_grads_finalize(const float *g32, float scale, void *g16, uint64_t n_padded, double *partials,
                                  double *out_sumsq, cudaStream_t st, int *n_launches);

// p16 = RNE_bf16(p)
cudaError_t launch_regen_bf16(const float *p, void *p16, uint64_t n_padded, cudaStream_t st);

// a6, bulk-kernel mode: src[k] = device-visible address of plane k inside the host slot's payload (p ‖ m ‖ v),
// dst[k] the live plane it restores; n = 3 for the one-phase restore, {p} then {m, v} for the two-phase one.
// p16 != nullptr: the bf16 copy is regenerated from plane 0 (must be p); kModeF32 shards have no bf16 copy.
struct RestorePlanes {
    const float *src[3];
    float *dst[3];
    int n;
};
// max_ctas: persistent CTAs (96 KB of shared memory each).  The link, not the SMs, is the bound, so a handful keeps it
// busy; the two-phase restore runs its second phase on few CTAs so that the recomputed iteration's kernels keep the SMs.
cudaError_t launch_restore_bulk(const RestorePlanes &pl, void *p16, uint64_t n_padded, int max_ctas, cudaStream_t st);

}  // namespace phx
