/*
 * phx.h — C ABI of the PHOENIX in-memory optimizer-state checkpoint hot path on B200 (sm_100a).
 *
 * What it is: the per-iteration replication of a data-parallel rank's sharded optimizer
 * state (fp32 master weights, Adam first/second moments, step count) taken INSIDE the
 * distributed-optimizer AdamW update, and the restore of a lost shard from that replica.
 * Paper: /root/reference/PAPER.md §V-B "Asynchronous Offload Pipeline" (lines 143-154),
 * §VI-A "In-Memory State Protection" (208-226), §V-C recovery stage 3 (171),
 * §VI-E/F restoration and resume (248-254).  The peer node's memory of the paper is stood
 * in for by a pinned host replica on the same box (BASELINE.json:north_star).
 *
 * General conventions
 *   - Every function returns int: PHX_OK (0) or a negative PHX_ERR_*.  No exceptions, no
 *     aborts, nothing is printed.
 *   - Pointers named d_* are DEVICE pointers (HBM of the current CUDA device), h_* are HOST
 *     pointers.  Replica memory must be pinned (page-locked) and mapped: the restore kernel
 *     reads it directly over the host link.  All buffers are owned by the caller (allocate
 *     them with any CUDA allocator, e.g. torch); the library never frees them and only owns
 *     small internals (events, a few KB of device scratch, one fp64 reduction partial per 16384 elements).
 *   - Streams are cudaStream_t passed as void*.  Calls that take a stream only ENQUEUE work;
 *     they never block the host on the device unless stated.  The three hot calls
 *     (phx_step_and_snapshot, phx_snapshot_flush_async, phx_restore / phx_restore_async) never do.  Host-blocking by
 *     contract: phx_snapshot_wait*, phx_restore_from / phx_replica_inspect (a blocking 512-byte read
 *     of a FOREIGN replica's envelopes), phx_last_clip, phx_graph_begin / phx_graph_end (mode
 *     switches), phx_shard_destroy.  Ordering between the compute stream and the flush stream
 *     is by library-owned events.  One host thread uses a handle at a time.
 *   - There is deliberately no fallback: a device that is not compute capability 10.x gives
 *     PHX_ERR_UNSUPPORTED_DEVICE at phx_shard_bind.
 *   - A shard belongs to the device that is current at phx_shard_bind.  Bind checks with
 *     cudaPointerGetAttributes that every d_* pointer is device (or managed) memory of THAT device
 *     (PHX_ERR_INVALID_ARG otherwise: a host pointer would fault asynchronously, far from the call) and that
 *     h_replica is pinned, mapped host memory.  The hot calls (step, flush, restore, their graph forms) return
 *     PHX_ERR_WRONG_DEVICE when another device is current.
 *
 * Memory layout (all little-endian, unit-stride)
 *   live state   d_p, d_m, d_v : float[n_padded]; d_p_bf16 : bf16[n_padded];
 *                d_grads_bf16  : bf16[n_padded] (read-only).  Lanes [n, n_padded) are padding:
 *                they must be zero in p, m, v and grads and the update keeps them exactly zero.
 *                Bases must be 256-byte aligned.
 *   snapshot     one packed contiguous buffer of snapshot_bytes =
 *                256 + 12*n_padded bytes:   header[256] ‖ p[n_padded] ‖ m[n_padded] ‖ v[n_padded]
 *   staging      d_staging : staging_depth snapshot slots, slot s at byte s*slot_stride
 *                (slot_stride = snapshot_bytes rounded up to 256).  Step k writes slot k mod depth.
 *   replica      h_replica : 2 snapshot slots at the same stride (ping-pong):
 *                the snapshot of step k lands in host slot k mod 2.
 *   header       phx_snapshot_header_t below — the paper's "metadata envelope (step index,
 *                parallelism configuration, RNG states)".
 */
#ifndef PHX_H
#define PHX_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PHX_API __attribute__((visibility("default")))

/* ---- errors ---------------------------------------------------------------------------- */
enum {
    PHX_OK = 0,
    PHX_ERR_INVALID_ARG = -1,
    PHX_ERR_ALIGNMENT = -2,           /* a bound pointer is not 256-byte aligned (d_p_bf16: 128) */
    PHX_ERR_NOT_BOUND = -3,           /* phx_shard_bind has not been called                      */
    PHX_ERR_STEP_ORDER = -4,          /* step != last_step + 1 (I4 step atomicity) */
    PHX_ERR_NO_FLUSH_PENDING = -5,    /* flush requested but no un-flushed snapshot exists       */
    PHX_ERR_NO_COMMITTED_SNAPSHOT = -6,
    PHX_ERR_LAYOUT_MISMATCH = -7,     /* replica belongs to another logical shard */
    PHX_ERR_CORRUPT_SLOT = -8,        /* reserved: both slots carry a header that fails checks   */
    PHX_ERR_CUDA = -9,                /* see phx_last_cuda_error                                  */
    PHX_ERR_UNSUPPORTED_DEVICE = -10, /* not compute capability 10.x; there is no fallback       */
    PHX_ERR_SNAPSHOT_DISABLED = -11,  /* flush/restore asked of a shard created with snapshots off */
    PHX_ERR_NOMEM = -12,
    PHX_ERR_PARAMS_NOT_READY = -13,   /* full-rank-state flush before phx_params_ready for that step  */
    PHX_ERR_GRAPH_MODE = -14,         /* eager call between phx_graph_begin/end, or a phx_graph_* call outside them */
    PHX_ERR_TOO_LARGE = -15,          /* phx_grad_sumsq_no_alloc: more elements than its built-in scratch serves */
    PHX_ERR_WRONG_DEVICE = -16        /* the current CUDA device is not the one the shard was bound on         */
};

/* ---- types ----------------------------------------------------------------------------- */
typedef struct phx_shard phx_shard_t; /* opaque */

/* One entry per tensor the rank holds after TP/PP slicing, in flattening order. */
typedef struct {
    uint64_t numel;
    uint32_t tensor_id;
    uint32_t flags; /* PHX_TENSOR_* bits; hashed into the layout hash */
} phx_tensor_desc_t;
/* Decay groups (reading R5b): a tensor flagged PHX_TENSOR_NO_DECAY (biases,
 * norm weights — the usual AdamW parameter groups) takes weight decay 0: decay = 1.0f for its elements,
 * so its trajectory equals a wd = 0 run bit for bit.  All other bits are reserved (must be 0). */
enum { PHX_TENSOR_NO_DECAY = 1u };

enum { PHX_SYNC_STRICT = 0, PHX_SYNC_RELAXED = 1 };
enum { PHX_RESTORE_COPY_ENGINE = 0, PHX_RESTORE_BULK_KERNEL = 1 };
enum { PHX_SNAPSHOT_STAGED = 0, PHX_SNAPSHOT_DIRECT = 1 };
/* PHX_PRECISION_BF16_GRADS (default, BASELINE.json:north_star): fp32 state, bf16 gradients, bf16 model-param
 * copy.  PHX_PRECISION_FP32: the precision the paper evaluates — "all parameters, main
 * gradients and optimizer states ... use torch.float32 ... BF16 and FP16 disabled": the
 * gradients are float[n_padded], there is no bf16 copy (d_p_bf16 may be NULL) and the fused kernel moves
 * 16 B read + 24 B written per element (12 written with snapshots off). */
enum { PHX_PRECISION_BF16_GRADS = 0, PHX_PRECISION_FP32 = 1 };
/* What the LOCAL host slots hold (the payloads are asymmetric by design).
 * PHX_PAYLOAD_OPTIMIZER (default): envelope ‖ p ‖ m ‖ v — the H2H payload, which is what the
 * host replica holds when it stands in for the peer (BASELINE.json:north_star).
 * PHX_PAYLOAD_FULL_RANK_STATE: the D2H payload of PAPER.md:145 — "the optimizer-state shard, the local
 * model-parameter shard, and a metadata envelope" — envelope ‖ p ‖ m ‖ v ‖ W, where W is the rank's
 * model-parameter buffer (see phx_shard_bind_params), so that a transient GPU fault is recovered in place
 * "without any network transfer".  Ring peers still receive the optimizer-only snapshot. */
enum { PHX_PAYLOAD_OPTIMIZER = 0, PHX_PAYLOAD_FULL_RANK_STATE = 1 };

/* Any field left 0 takes its default; cfg == NULL means all defaults. */
typedef struct {
    uint32_t tp_size, tp_rank, pp_size, pp_rank; /* logical identity only; sizes default 1      */
    uint32_t staging_depth;   /* 1..4 device staging slots; default 2                            */
    uint32_t sync_mode;       /* PHX_SYNC_STRICT (default): step k+1 waits for commit(k) — the
                                 paper's single sync point, replay <= 1 step.
                                 PHX_SYNC_RELAXED: step k+1 waits only until staging slot
                                 (k+1) mod depth has been drained, replay <= depth steps.        */
    uint64_t chunk_bytes;     /* D2H chunk size (any size, rounded up to 256 B; 4 MiB..256 MiB is the
                                 useful range); default 32 MiB (measured on c2..c5: 99.3 % of the pinned
                                 link rate against 95.5 % at 8 MiB, exposed time the same within run-to-run
                                 noise)                                                */
    uint32_t snapshot_disabled; /* 1: plain AdamW + bf16 copy, no staging stores (the paper's
                                 "mechanism disabled" baseline)                     */
    uint32_t restore_mode;    /* PHX_RESTORE_COPY_ENGINE (default, measured faster) | PHX_RESTORE_BULK_KERNEL */
    float max_grad_norm;      /* > 0: clip by the shard-local gradient norm before the step       */
    uint32_t snapshot_source; /* PHX_SNAPSHOT_STAGED (default): the fused kernel also writes the packed
                                 snapshot into a device staging slot, which the flush drains (the live state
                                 may move on at once; needed for PHX_SYNC_RELAXED).
                                 PHX_SNAPSHOT_DIRECT: no staging buffer and no staging stores — the flush DMAs
                                 the live p, m, v planes themselves.  Sound because under PHX_SYNC_STRICT the
                                 next step's kernel waits for commit(k) before it mutates the protected state
                                 (exactly the paper's sync point); requires PHX_SYNC_STRICT.
                                 The kernel then moves 28 B/element instead of 40.                           */
    uint32_t precision;       /* PHX_PRECISION_BF16_GRADS (default) | PHX_PRECISION_FP32                   */
    uint32_t payload;         /* PHX_PAYLOAD_OPTIMIZER (default) | PHX_PAYLOAD_FULL_RANK_STATE (local slots) */
    uint32_t reserved[2];
} phx_config_t;

typedef struct {
    uint64_t n;              /* real fp32 elements owned by this rank                             */
    uint64_t n_padded;       /* plane length: total padded to a multiple of 64*dp_size, / dp_size */
    uint64_t total_numel;    /* sum of layout numel                                               */
    uint64_t shard_begin;    /* dp_rank * n_padded: start of the rank's range in the flat space   */
    uint64_t layout_hash;    /* FNV-1a 64 over the tensor descriptors and dp/tp/pp sizes+tp/pp rank */
    uint64_t snapshot_bytes; /* 256 + 12*n_padded                                                 */
    uint64_t slot_stride;    /* snapshot_bytes rounded up to 256                                  */
    uint32_t n_segments, staging_depth;
    uint32_t dp_size, dp_rank;
    /* local host slots (h_replica): equal to snapshot_bytes / slot_stride under PHX_PAYLOAD_OPTIMIZER;
     * under PHX_PAYLOAD_FULL_RANK_STATE host_snapshot_bytes = snapshot_bytes + param_bytes */
    uint64_t host_snapshot_bytes, host_slot_stride;
    uint64_t param_bytes;    /* dp_size * n_padded * (2 | 4): size of the model-parameter buffer W   */
} phx_shard_info_t;

/* The 256-byte metadata envelope at the front of every snapshot slot. */
typedef struct {
    uint8_t magic[8];       /* "PHXSNAP1"                                                         */
    uint32_t version;       /* 1                                                                  */
    uint32_t header_bytes;  /* 256                                                                */
    uint64_t seq_begin;     /* == step                                                            */
    uint64_t step;          /* state in this slot is the state AFTER optimizer step `step`        */
    uint64_t n, n_padded, total_numel, shard_begin, layout_hash;
    uint32_t dp_size, dp_rank, tp_size, tp_rank, pp_size, pp_rank;
    uint64_t chunk_bytes;
    uint32_t user_len;      /* bytes used of user[]                                               */
    uint32_t payload;       /* 0: p ‖ m ‖ v follow; 1 | elem_bytes << 8: p ‖ m ‖ v ‖ W follow (full rank state) */
    uint8_t user[128];      /* opaque caller blob (RNG states...), restored bit-exactly           */
    uint64_t header_hash;   /* FNV-1a 64 of bytes [0, 240)                                        */
    uint64_t seq_end;       /* == seq_begin once the slot is committed; written last              */
} phx_snapshot_header_t;

/* ---- a0: shard definition (host only; works without a GPU) -------------------------------
 * Flatten the tensor list in order, pad the total up to a multiple of 64*dp_size, cut dp_size
 * equal contiguous ranges; this rank owns [dp_rank*L, (dp_rank+1)*L) ("sharded model and
 * optimizer states"; ZeRO-2 distributed optimizer).  A tensor may
 * straddle ranks; the segment table records the pieces.  layout is copied. */
PHX_API int phx_shard_create(const phx_tensor_desc_t *layout, size_t n_tensors, uint32_t dp_size,
                             uint32_t dp_rank, const phx_config_t *cfg, phx_shard_t **out);
PHX_API int phx_shard_destroy(phx_shard_t *s); /* waits for in-flight flushes, frees internals */
PHX_API int phx_shard_info(const phx_shard_t *s, phx_shard_info_t *out);
/* Fills up to cap entries (all four arrays have cap entries); entry i is the i-th piece of
 * the rank's range: tensor_id, offset inside that tensor, offset inside the shard, length. */
PHX_API int phx_shard_segments(const phx_shard_t *s, uint32_t *tensor_id, uint64_t *off_in_tensor,
                               uint64_t *off_in_shard, uint64_t *len, uint32_t cap);

/* ---- binding memory -----------------------------------------------------------------------
 * d_staging: staging_depth * slot_stride bytes of device memory (may be NULL iff snapshots are
 * disabled or snapshot_source is PHX_SNAPSHOT_DIRECT).  h_replica: 2 * slot_stride bytes of pinned, mapped
 * host memory (may be NULL if snapshots are disabled or only peer replicas are used, see
 * phx_shard_bind_peers; phx_snapshot_flush_async / phx_restore then return PHX_ERR_NOT_BOUND).
 * Requires a CUDA device of compute capability 10.x. */
/* d_p_bf16 may be NULL iff precision is PHX_PRECISION_FP32; it needs 128-byte alignment only, so that it can be
 * the rank's range inside its model-parameter buffer W (W + dp_rank * n_padded elements, §8(f3)). */
PHX_API int phx_shard_bind(phx_shard_t *s, float *d_p, float *d_m, float *d_v, void *d_p_bf16,
                           void *d_staging, void *h_replica);
/* Declare the bound p, m, v to be the state after optimizer step `step` (0 at initialisation)
 * and regenerate d_p_bf16 = RNE_bf16(p) on `stream`. */
PHX_API int phx_shard_set_state(phx_shard_t *s, uint64_t step, void *stream);
/* Opaque blob (<= 128 bytes) copied into the header of every later snapshot.  PHX_ERR_GRAPH_MODE between
 * phx_graph_begin and phx_graph_end (the envelope template then lives on the device): use
 * phx_graph_set_user_metadata there. */
PHX_API int phx_set_user_metadata(phx_shard_t *s, const void *blob, uint32_t len);

/* ---- a1+a2+a3: fused AdamW step + snapshot -------------------------------------------------
 * Enqueues on `stream`:
 *   a1 (only if max_grad_norm > 0): S = sum g^2 in fp64 by a fixed tree whose shape depends on n alone, clip
 *      coefficient c = fp32(min(1, max_grad_norm / (sqrt(S) + 1e-6))) left in device memory;
 *   a2: wait (stream-side, not host-side) until the previous snapshot is committed (strict) or
 *      the staging slot about to be written has been drained (relaxed) — PAPER.md:226;
 *   a3: ONE kernel making one pass over the shard.  Per element, in fp32 with every operation
 *      individually rounded (no FMA contraction, no flush-to-zero, IEEE sqrt and divide):
 *        g = widen(g_bf16) * c;  p1 = p * decay;  m' = beta1*m + omb1*g;
 *        v' = beta2*v + omb2*(g*g);  d = sqrt(v')/sbc2 + eps;  p' = p1 - ss*(m'/d)
 *      with decay = 1 - lr*wd, omb1 = 1 - beta1, omb2 = 1 - beta2, ss = lr/(1 - beta1^step),
 *      sbc2 = sqrt(1 - beta2^step) computed on the host in double and rounded once to fp32.
 *      It writes p', m', v' to the live arrays, RNE_bf16(p') to d_p_bf16, and the same p', m',
 *      v' bits plus the header into staging slot `step mod depth` ("packed into a contiguous
 *      buffer") — the snapshot costs no extra read pass and no extra kernel.
 * `step` is the 1-based index of the update and must equal last_step + 1.
 * Caller's contract (strict mode, "replay <= 1 step"): flush snapshot k (phx_snapshot_flush_async
 * and/or phx_snapshot_flush_peers_async) BEFORE enqueuing step k+1 — the sync point can only wait for a flush
 * that has been enqueued.  A step that finds its predecessor's snapshot never flushed goes ahead (that snapshot
 * is superseded, replay grows by one step) and counts it: phx_dropped_snapshots.
 * d_grads: bf16[n_padded] (PHX_PRECISION_BF16_GRADS) or float[n_padded] (PHX_PRECISION_FP32: first line
 * g = g_f32 * c, no bf16 copy is written, the sum of squares uses exact fp64 squares of the fp32 values).
 * Elements of tensors flagged PHX_TENSOR_NO_DECAY use decay = 1.0f.
 * Traffic: reads 14 B/element, writes 26 B/element (14 with snapshots disabled); FP32: 16 + 24 (12). */
PHX_API int phx_step_and_snapshot(phx_shard_t *s, const void *d_grads, float lr, float beta1,
                                  float beta2, float eps, float wd, uint64_t step, void *stream);

/* ---- a4+a5: asynchronous chunked flush of the newest staged snapshot ------------------------
 * Enqueues on `side_stream` (a copy-engine stream, "dedicated CUDA stream"):
 * wait for the step's kernel; invalidate the host slot's header; copy the payload in
 * chunk_bytes pieces; copy the header last (= commit: seq_end lands last).  The other host
 * slot keeps the previous committed snapshot throughout. */
PHX_API int phx_snapshot_flush_async(phx_shard_t *s, void *side_stream);
/* Host-blocking wait until the snapshot of `step` is committed (tests, shutdown). */
PHX_API int phx_snapshot_wait(phx_shard_t *s, uint64_t step);
/* Non-blocking: newest snapshot known committed (by completed flush events); *slot = host slot
 * index, or PHX_ERR_NO_COMMITTED_SNAPSHOT. */
PHX_API int phx_snapshot_query(phx_shard_t *s, uint64_t *newest_committed_step, int *slot);
/* Fault injection for tests: the NEXT flush copies only `payload_chunks` payload
 * chunks and never commits; the slot stays torn.  payload_chunks < 0 clears the hook. */
PHX_API int phx_fault_inject_torn_flush(phx_shard_t *s, int64_t payload_chunks);

/* ---- a6: restore ---------------------------------------------------------------------------
 * ENQUEUE-ONLY: the host never waits for the device.  Chooses between the two host slots the valid
 * one (magic, version, header hash, seq_begin == seq_end) with the largest step, refuses it if
 * its logical identity (layout hash, dp/tp/pp coordinates, n) differs from this shard's, and
 * enqueues on `stream` the rebuild of the live shard: p, m, v from the slot and d_p_bf16 =
 * RNE_bf16(p).  The envelope that decides is the one IN the pinned slot (plain host read) for every slot
 * this handle is not writing at that moment; for a slot whose flush by THIS handle is still in flight the
 * handle's own record of the envelope it sent decides (a flush cannot tear unless told to, and a torn one is
 * skipped), and `stream` waits for that flush's event before the copies.  `stream` also waits for whatever of
 * this handle may still touch the live planes (the newest step's kernel, a direct-source flush, a
 * publication), so a restore issued while step k+1's kernel and flush(k) are in flight is well ordered.  PHX_RESTORE_COPY_ENGINE: three H2D copies straight into the live planes (the packed
 * layout is planar, so no unpack pass is needed) plus a bf16 regeneration kernel;
 * PHX_RESTORE_BULK_KERNEL: one kernel pulls the replica straight from mapped host memory with 1-D
 * bulk async (TMA) loads into shared memory and writes all four arrays.  Both are bit-exact; the
 * copy engine reaches 99.5 % of the pinned H2D peak, SM/TMA-issued PCIe reads 92 % (128-byte
 * read requests), hence the default.  Depends on
 * nothing in device memory.  Afterwards last_step = header.step, so the caller re-issues step
 * last_step + 1 with the same gradients (recompute of the in-flight step).
 * A fresh handle created with the same layout/coordinates and bound to the same replica can
 * restore too (a replacement rank assuming the failed rank's role). */
PHX_API int phx_restore(phx_shard_t *s, void *stream, uint64_t *restored_step);
/* a6 in TWO PHASES (reading R37).  "Model parameters are reconstructed ... while optimizer state is
 * restored from in-memory replicas ... Finally, execution resumes from the last completed step" (PAPER.md:171,
 * §V-C): the recomputed iteration's forward/backward reads only the model parameters; the moments are first read
 * by its optimizer step.  phx_restore_async makes the same choice of slot, identity check and hazard ordering as
 * phx_restore (and only enqueues), but runs everything on `side_stream` in the order
 *     optimizer-only payload:  p -> model-param copy (bf16 regeneration)  == "parameters ready";   m -> v  == "state ready"
 *     full rank state:         W (alone: the rank's own range of W IS its model-param copy, and the forward/backward
 *                              reads nothing else)                          == "parameters ready";   p -> m -> v  == "state ready"
 * (PHX_RESTORE_BULK_KERNEL: two launches of the bulk kernel, the second — beside the recomputed iteration — on four
 * persistent CTAs, which already saturate the host link and leave the other SMs to the compute).
 * phx_restore_wait_params makes `stream` wait (stream-side) until the parameters are in place, after which the
 * forward/backward of the recomputed iteration may be enqueued on it; two thirds of the host-link transfer then
 * hide behind that compute.  The next phx_step_and_snapshot (any stream) waits for "state ready" by itself, and so do
 * phx_restore*, phx_graph_begin and the publication calls; the final state is bit-identical to phx_restore's.
 * On return last_step = header.step.  A no-op wait when no two-phase restore is outstanding. */
PHX_API int phx_restore_async(phx_shard_t *s, void *side_stream, uint64_t *restored_step);
PHX_API int phx_restore_wait_params(phx_shard_t *s, void *stream);
/* Copies the user blob of the slot the last phx_restore used. */
PHX_API int phx_restored_user_metadata(const phx_shard_t *s, void *blob, uint32_t cap, uint32_t *len);

/* ---- peer replication around the data-parallel ring ------------------------
 * The paper's H2H phase: the packed optimizer snapshot (envelope ‖ p ‖ m ‖ v — no
 * model parameters) is sent to the ring peer, "the rank sharing the same
 * tensor-parallel and pipeline-parallel positions but with a different data-parallel index"; with
 * multi-peer replication to k distinct DP peers.  On a B200 NVLink 5 / NVSwitch box the
 * peer's memory is reached directly: the peer process allocates a RECEIVED BUFFER (two snapshot slots at
 * slot_stride, "committed / receiving", Fig. 5, 224) in its GPU's HBM, exports it over CUDA
 * IPC, and the owner's copy engine writes the staging slot (or, in PHX_SNAPSHOT_DIRECT, the live planes)
 * into it over NVLink on a dedicated stream — same protocol as the local pair: header invalidated,
 * payload in chunk_bytes pieces, valid header last, slot = step mod 2.  No SM is involved and nothing is
 * added to the critical path; pushing the snapshot stores themselves over NVLink from the fused kernel
 * would put 12 B/element at ~0.9 TB/s (2.2 ms at c2) on it instead of 0.3 ms.
 * The sync point of phx_step_and_snapshot (a2) also waits for the peer flush: "guarantees the
 * peer-resident replica is fully committed before the optimizer mutates the protected state"
 * (PAPER.md:226). */
#define PHX_MAX_PEERS 4
#define PHX_IPC_HANDLE_BYTES 64
/* Ring peer j of rank r: (r + j) mod dp_size; j = 1..k are the ranks that hold r's replicas, j = -1..-k the
 * ranks whose replicas r holds.  |j| must be in [1, dp_size - 1] (k distinct peers need k <= D - 1). */
PHX_API int phx_ring_peer(uint32_t dp_size, uint32_t dp_rank, int32_t j, uint32_t *peer);
/* Topology-aware placement ("place the k replicas on nodes under k distinct switches or racks, ensuring
 * that a single infrastructure event affects at most one copy of any given shard"; reading R38): with
 * domain_of_rank[q] = the failure domain (switch, rack, node, ...) of DP rank q, peers[0..k) receives the k nearest
 * ranks in ring order (dp_rank + 1, dp_rank + 2, ...) whose domains differ from the owner's and from one another, so
 * that the k + 1 copies of the shard sit under k + 1 distinct domains.  k <= min(PHX_MAX_PEERS, dp_size - 1);
 * PHX_ERR_INVALID_ARG when fewer than k + 1 distinct domains exist.  One rank per domain gives phx_ring_peer's ring.
 * Host arithmetic only; the buffers of whichever ranks are chosen are bound with phx_shard_bind_peers as before. */
PHX_API int phx_ring_peers_topology_aware(uint32_t dp_size, uint32_t dp_rank, uint32_t k, const uint32_t *domain_of_rank,
                                          uint32_t *peers);
/* Received-buffer memory: a zeroed device allocation of its own (cudaMalloc), so that it can be exported
 * over CUDA IPC; owned by the caller, freed with phx_peer_buffer_free. */
PHX_API int phx_peer_buffer_alloc(uint64_t bytes, void **d_buf);
PHX_API int phx_peer_buffer_free(void *d_buf);
/* CUDA IPC plumbing (cudaIpcGetMemHandle / cudaIpcOpenMemHandle with lazy peer access / Close): export a
 * buffer allocated with phx_peer_buffer_alloc; open it in ANOTHER process of the same node. */
PHX_API int phx_ipc_export(void *d_buf, uint8_t handle[PHX_IPC_HANDLE_BYTES]);
PHX_API int phx_ipc_open(const uint8_t handle[PHX_IPC_HANDLE_BYTES], void **d_buf);
PHX_API int phx_ipc_close(void *d_buf);
/* d_peer_replicas[j-1]: device-addressable address of the received buffer (2 * slot_stride bytes) that ring
 * peer j keeps for this rank; k <= min(PHX_MAX_PEERS, dp_size - 1) distinct buffers; k = 0 unbinds.
 * h_replica of phx_shard_bind may be NULL when only peers are used. */
PHX_API int phx_shard_bind_peers(phx_shard_t *s, void *const *d_peer_replicas, uint32_t k);
/* Enqueues the replication of the newest snapshot to all k peers.  k = 1: on `peer_stream`.  k > 1: on k
 * library-owned copy streams forked from and joined back into `peer_stream` (one copy engine / NVSwitch path
 * per peer; `peer_stream` observes the completion of all of them).  Independent of phx_snapshot_flush_async: either or both
 * may be called after a step, on different streams, and overlap (PCIe and NVLink are separate links). */
PHX_API int phx_snapshot_flush_peers_async(phx_shard_t *s, void *peer_stream);
/* Host-blocking wait until the peer replication of `step` is committed on every peer. */
PHX_API int phx_snapshot_wait_peers(phx_shard_t *s, uint64_t step);
/* Fault injection: the NEXT replication to ring peer `peer_j` (1-based) stops after
 * `payload_chunks` payload chunks and never commits. */
PHX_API int phx_fault_inject_torn_peer_flush(phx_shard_t *s, uint32_t peer_j, int64_t payload_chunks);
/* What a replica buffer (device, peer-mapped or pinned host memory) holds: both headers and whether each
 * passes the commit rule.  Host-blocking.  A holder uses it to answer "which logical shard, which step"
 * when sources and replacements are matched by logical shard identity. */
PHX_API int phx_replica_inspect(const void *replica, uint64_t slot_stride, phx_snapshot_header_t out[2], int valid[2]);
/* a6 from a replica held elsewhere (recovery stage 3: "optimizer state is restored from
 * in-memory replicas"): `replica` is any device-accessible address of two snapshot slots — the surviving
 * holder's received buffer opened over IPC, a device buffer, or pinned mapped host memory.  Same slot
 * selection, identity check, restore modes and postconditions as phx_restore.  The replica is foreign (this
 * handle has no commit record of it), so the two envelopes are read with a BLOCKING 512-byte copy — the one
 * documented exception to "restore only enqueues". */
PHX_API int phx_restore_from(phx_shard_t *s, const void *replica, void *stream, uint64_t *restored_step);

/* ---- model-parameter publication and reconstruction ---------------------------
 * In the ZeRO-2 distributed optimizer every DP rank of one TP/PP coordinate holds the same
 * model parameters W for that partition: the flat padded space of a0 in the model dtype (bf16; float in
 * PHX_PRECISION_FP32), dp_size * n_padded elements, rank r's range at element offset r * n_padded.  After
 * the step each rank has updated only its own range and the ranges are all-gathered (R29).
 * PHX_PUBLISH_FUSED: the step → all-gather pair is ONE kernel: phx_step_and_snapshot's fused kernel stores
 * every element's model-param copy not only to d_p_bf16 (the caller points it at its own W + r * n_padded)
 * but also into the same range of each bound peer buffer (peer HBM over NVLink 5 / NVSwitch, mapped with
 * phx_ipc_open) — no separate all-gather kernel, no extra read of the copy.
 * PHX_PUBLISH_COPY_ENGINE: the kernel is unchanged and phx_publish_params_async pushes the range to the
 * peers with `count` copy-engine copies on a side stream (after the step's kernel).
 * d_param_bufs[i]: base address of another rank's W (device-addressable); count <= PHX_MAX_PARAM_PEERS.
 * In PHX_PRECISION_FP32 the published values are the fp32 parameters p themselves. */
#define PHX_MAX_PARAM_PEERS 15
enum { PHX_PUBLISH_FUSED = 0, PHX_PUBLISH_COPY_ENGINE = 1 };
PHX_API int phx_shard_bind_param_peers(phx_shard_t *s, void *const *d_param_bufs, uint32_t count, uint32_t mode);
PHX_API int phx_publish_params_async(phx_shard_t *s, void *stream);
/* R30: a replacement rank reconstructs its model parameters from a healthy DP rank
 * of the same TP/PP coordinate: one copy of the whole buffer W (dp_size * n_padded model-dtype elements)
 * from `d_src_param_buf` (peer HBM) into `d_dst_param_buf`. */
PHX_API int phx_params_restore_from(phx_shard_t *s, const void *d_src_param_buf, void *d_dst_param_buf, void *stream);

/* ---- full rank-state local snapshot and in-place recovery ---------------------
 * With cfg.payload = PHX_PAYLOAD_FULL_RANK_STATE the local host slots hold the D2H payload of
 * envelope(payload = 1 | elem_bytes << 8) ‖ p ‖ m ‖ v ‖ W, host_snapshot_bytes long at
 * host_slot_stride (h_replica of phx_shard_bind must then hold 2 * host_slot_stride bytes).  W is the
 * model-parameter buffer the rank holds for its TP/PP partition (the buffer of §8(f3): dp_size * n_padded
 * elements of the model dtype, rank r's range at element r * n_padded); in PHX_PRECISION_BF16_GRADS
 * d_p_bf16 of phx_shard_bind must be the rank's own range inside it (d_W + dp_rank * n_padded elements).
 * Staging slots and ring-peer slots keep the optimizer-only layout.
 *
 * Protocol per step k:  phx_step_and_snapshot(k)  →  [the partition's all-gather of step k lands in W]  →
 * phx_params_ready(stream): the caller declares, in `stream` order, that W now holds every rank's
 * parameters after step k  →  phx_snapshot_flush_async: waits for the step's kernel AND for that
 * declaration (PHX_ERR_PARAMS_NOT_READY if it was not made for step k), then header invalidated, W in
 * chunk_bytes pieces, p ‖ m ‖ v in chunk_bytes pieces, valid header last (W first: it is the part other
 * ranks overwrite at their next publication).  phx_fault_inject_torn_flush counts chunks in that order.
 * phx_params_guard(stream): `stream` waits until the newest flush has finished READING W — to be enqueued
 * ahead of whatever lets other ranks publish step k+1 into this rank's W (handing this rank's gradients to
 * the reduce-scatter of iteration k+1; a local copy-engine publication).  The rank's own step k+1 is
 * covered by phx_step_and_snapshot: the strict sync point waits for the whole flush, and under
 * PHX_SYNC_RELAXED the step additionally waits until the newest flush has finished reading W (its own range
 * of W is d_p_bf16, which the kernel rewrites).
 *
 * phx_restore on such a shard is the in-place recovery: p, m, v AND W come back from
 * the rank's own host slot (newest valid slot whose payload word and identity match), nothing is read from
 * any other rank; the rank's own range of W equals RNE_bf16(p) again by construction.  Copy engine only
 * (cfg.restore_mode is ignored for the W part).  phx_restore_from (a peer's optimizer-only replica) and
 * phx_params_restore_from remain the permanent-failure path. */
PHX_API int phx_shard_bind_params(phx_shard_t *s, void *d_W);
PHX_API int phx_params_ready(phx_shard_t *s, void *stream);
PHX_API int phx_params_guard(phx_shard_t *s, void *stream);

/* ---- the DP-global gradient-norm clip (the one scalar exchange of the path) -------
 * "Global grad-norm clip 1.0" (BASELINE.json:configs[2]); "all-reduce of sum g^2 for
 * the global clip".  With dp_size > 1 the norm that decides the clip is the norm of the WHOLE gradient:
 *     S = sum over ranks r of S_r,  S_r = sum_i g_{r,i}^2,  c = fp32(min(1, max_grad_norm/(sqrt(S)+1e-6)))
 * and every rank applies the same c (oracle/global_clip.py).  a1 is therefore split in two around the
 * caller's exchange of D doubles (NCCL all-gather on the same stream; 8*D bytes):
 *
 *   phx_grad_sumsq_async(s, d_grads, d_out, stream)   S_r of this rank's gradient shard (same kernels, same
 *        fixed fp64 tree as the local a1) written to the caller-owned device double *d_out
 *        (8-byte aligned).  Needs a bound shard; does not touch the optimizer state or the step counter.
 *        It uses the handle's a1 reduction scratch: enqueue it on the SAME stream as the step that follows.
 *   [caller: all-gather the D values into a device array ordered by dp_rank]
 *   phx_set_clip_partials(s, d_partials, count)       ONE-SHOT: the next phx_step_and_snapshot skips its own
 *        sum-of-squares pass and takes S = d_partials[0] + ... + d_partials[count-1] (fixed tree, so every
 *        rank that was handed the same array gets the same bits; count in 1..1024; the array is read on the
 *        step's stream, in stream order, and must stay valid until that kernel has run).  count = 1 with an
 *        already all-reduced scalar is equally valid.  Requires cfg.max_grad_norm > 0, else
 *        PHX_ERR_INVALID_ARG.  Cleared by the step that consumes it and by phx_restore* (the recompute of
 *        the in-flight step supplies its partials again).  d_partials = NULL clears it.
 * With count = 1 and d_partials = the rank's own S_r the coefficient is bit-identical to the local a1. */
PHX_API int phx_grad_sumsq_async(phx_shard_t *s, const void *d_grads, double *d_out, void *stream);
PHX_API int phx_set_clip_partials(phx_shard_t *s, const double *d_partials, uint32_t count);

/* ---- a1 for callers that must not allocate device memory -------------------------------------------
 * phx_grad_sumsq_no_alloc: the same S_r = sum_i g_i^2 as phx_grad_sumsq_async (same kernels, same fixed fp64
 * tree, hence the same bits on the same gradients), but without a handle and without a single allocation:
 * it calls neither cudaMalloc nor cudaFree nor any routine that does.
 *
 * Who needs it.  phx_grad_sumsq_async wants a bound shard, and phx_shard_bind gets the reduction scratch from
 * cudaMalloc.  That is no option for (i) a trainer whose framework allocator already holds all of the GPU's
 * memory — an allocation made beside it fails, or robs the framework and surfaces as its out-of-memory error
 * later; (ii) code on the iteration's critical path — cudaMalloc and cudaFree synchronise the device, so one
 * call from a monitoring thread stalls the very flush/compute overlap this library exists for (PAPER.md:128,
 * 143); (iii) the fault-handling side, which wants a rank's gradient norm at the moment the
 * allocator is least to be relied on.  For these callers the scratch is built into the library image.
 *
 * The limit.  The scratch is one statically declared device array of 65536 doubles = 512 KiB; EVERY GPU on
 * which the process uses libphx.so holds it from module load until the process exits, whether or not this call is
 * ever made.  It serves n_elems <= PHX_NO_ALLOC_MAX_ELEMS = 2^30 elements (one partial per 16384); a larger
 * n_elems returns PHX_ERR_TOO_LARGE and enqueues nothing.
 *
 * Arguments.  d_grads: device, read-only, 256-byte aligned; bf16[n_elems] if grads_fp32 == 0, float[n_elems]
 * if grads_fp32 == 1 (any other value: PHX_ERR_INVALID_ARG).  n_elems: > 0 and a multiple of 8 (a shard's
 * n_padded always is); padding lanes must be zero.  d_out: device double, 8-byte aligned, caller-owned, written in
 * `stream` order.  stream: cudaStream_t; the call only enqueues two kernels.  cuda_error: optional (may be NULL);
 * receives the cudaError_t when the result is PHX_ERR_CUDA, else 0.  Works on the CURRENT device, which must be
 * compute capability 10.x (PHX_ERR_UNSUPPORTED_DEVICE otherwise) and the one d_grads and d_out live on.
 *
 * Sharing.  There is ONE array per GPU for all callers and threads.  It keeps the previous call's contents; no
 * clearing is needed, because each call first overwrites exactly the entries it then reads.  Calls whose kernels
 * can overlap on one GPU (unordered streams) RACE on the array and return garbage: keep them on one stream or
 * order them with events.  The handle-based calls use their own scratch and are unaffected.
 *
 * First call.  The first call on each device looks up the array's device address (and thereby makes the driver
 * load the library's module on that device); it takes a process-wide mutex and is slower than the rest.  Make it
 * once per device BEFORE any stream capture begins. */
#define PHX_NO_ALLOC_MAX_ELEMS (1ull << 30)
PHX_API int phx_grad_sumsq_no_alloc(const void *d_grads, int grads_fp32, uint64_t n_elems, double *d_out,
                                    void *stream, int *cuda_error);

/* ---- SURVEY.md §8(f4), second half: the gradient producer's epilogue -------------------------------
 * "single-pass fusion of the sum-of-squares with the previous step's epilogue".  The
 * gradients of step k+1 do not exist while step k's kernel runs and the clip coefficient must be known before
 * the first element of step k+1 moves, so the one place where the norm costs no pass of its own is the
 * PRODUCER of the optimizer's gradients: the epilogue of the reduce-scatter of the binary32 main gradients
 * (ZeRO-2 distributed optimizer; "main gradients ... torch.float32").  One kernel,
 * one pass (4 B read + 2 B written per element; reading R34):
 *     g16_i = RNE_bf16(g32_i * scale)      one binary32 multiply (scale: gradient averaging; 1.0f exact), then
 *                                          the same rounding as the bf16 model-param copy
 *     *d_sumsq_out = sum_i widen(g16_i)^2  fp64, of the ROUNDED values, by the SAME fixed tree as a1 — the very
 *                                          number, bit for bit, a1 would compute from g16
 * d_main_grads_fp32: float[n_padded] (pad lanes zero), d_grads_bf16_out: bf16[n_padded], both 256-byte
 * aligned, not overlapping; d_sumsq_out: device double, 8-byte aligned.  Then
 *     phx_set_clip_partials(s, d_sumsq_out, 1);  phx_step_and_snapshot(s, d_grads_bf16_out, ...)
 * runs the step with NO sum-of-squares pass (40 instead of 42 B/element on the critical path).  It has a
 * reduction scratch of its own inside the handle (it may run on the producer's stream while a step with its own
 * a1 pass runs on another); two epilogues of one handle must be stream-ordered.  PHX_PRECISION_BF16_GRADS only. */
PHX_API int phx_grads_finalize_async(phx_shard_t *s, const float *d_main_grads_fp32, float scale,
                                     void *d_grads_bf16_out, double *d_sumsq_out, void *stream);

/* ---- the graph-capturable form of a1..a5 -----------------------------------------------------------
 * phx_step_and_snapshot carries per-step values (ss, sbc2, the envelope) as kernel parameters, so a captured
 * launch would replay a stale step.  Between phx_graph_begin and phx_graph_end the step index, the
 * hyperparameters, the derived scalars and the envelope live in a DEVICE-RESIDENT step block: a one-thread
 * prologue kernel advances the counter, derives the scalars in binary64 with individually rounded operations
 * (the same bits as the host path) and writes the envelope; the fused kernel reads the scalars from there.
 * Nothing per-step crosses the host, so  [compute window ‖ flush(k-1)] -> step k  can be captured once with
 * cudaStreamBeginCapture / torch.cuda.graph and replayed (the sync point is then an edge of the
 * graph).  The calls also work eagerly (same kernels), which is how a run enters and leaves.
 *
 *   phx_graph_begin(s, lr, beta1, beta2, eps, wd, stream)   mode switch (host-blocking: lands this handle's eager
 *        flushes), initialises the step block at last_step on `stream`.  An un-flushed eager snapshot becomes
 *        the first phx_graph_flush_async's work.  With PHX_PAYLOAD_FULL_RANK_STATE (§8(f4)) the protocol is
 *        the eager one with the same two calls, which become edges of the captured graph between begin and end:
 *        phx_params_ready(stream) before the flush of that step (else PHX_ERR_PARAMS_NOT_READY),
 *        phx_params_guard(stream) ahead of whatever overwrites W; a declaration made eagerly for a still
 *        pending snapshot carries over in both directions.
 *   phx_graph_set_hyper(...)                                 stream-ordered update of the hyperparameters (learning-
 *        rate schedules) between replays; not captured itself.
 *        PHX_ERR_INVALID_ARG if `stream` is being captured (its source is host memory of the call).
 *   phx_graph_set_user_metadata(s, blob, len, stream)        the same for the caller blob of the envelope (RNG states,
 *        PAPER.md:145): stream-ordered update of the device-resident envelope template; every snapshot whose
 *        prologue runs after it on `stream` carries the new blob (and so do the eager calls after
 *        phx_graph_end).  Call it between replays; not capturable (PHX_ERR_INVALID_ARG on a capturing stream).
 *   phx_graph_step_and_snapshot(s, d_grads, stream)          a1 (if configured) + a2 + prologue + a3, capturable.  The
 *        staging slot (issue index mod depth) and the host slot parity are fixed when the call is CAPTURED:
 *        a captured sequence must span a multiple of lcm(depth, 2) steps and be replayed from the step
 *        parity it was captured at; the prologue checks it on the device and phx_graph_end reports
 *        PHX_ERR_STEP_ORDER if a replay ever ran misaligned.
 *   phx_graph_flush_async(s, side_stream)                    a4 + a5 of the snapshot of the last ISSUED step,
 *        capturable.  Inside a capture `side_stream` must already belong to the capture (fork it from the
 *        capturing stream: record an event there, wait for it on side_stream); the next
 *        phx_graph_step_and_snapshot's sync point joins it back.
 *   phx_graph_end(s, &last_step)                             mode switch (cudaDeviceSynchronize): reads the device step
 *        counter, rebuilds the commit bookkeeping from the self-describing host slots; afterwards the eager
 *        calls continue at last_step + 1 and a still-staged newest snapshot can be flushed eagerly.
 * Eager calls (step, flush, restore, phx_set_user_metadata, phx_publish_params_async, phx_last_clip) return
 * PHX_ERR_GRAPH_MODE in between, phx_graph_* outside. */
PHX_API int phx_graph_begin(phx_shard_t *s, float lr, float beta1, float beta2, float eps, float wd, void *stream);
PHX_API int phx_graph_set_hyper(phx_shard_t *s, float lr, float beta1, float beta2, float eps, float wd, void *stream);
PHX_API int phx_graph_set_user_metadata(phx_shard_t *s, const void *blob, uint32_t len, void *stream);
PHX_API int phx_graph_step_and_snapshot(phx_shard_t *s, const void *d_grads, void *stream);
PHX_API int phx_graph_flush_async(phx_shard_t *s, void *side_stream);
/* §8(f1) in the graph form: replication of the last issued step's snapshot to the k bound ring peers, capturable
 * like phx_graph_flush_async (fork `peer_stream` from the capturing stream first; k > 1 fans out over the
 * library-owned per-peer streams inside the capture).  The sync point of the next step covers it. */
PHX_API int phx_graph_flush_peers_async(phx_shard_t *s, void *peer_stream);
PHX_API int phx_graph_end(phx_shard_t *s, uint64_t *last_step);

/* ---- introspection ---------------------------------------------------------------------- */
PHX_API int phx_last_step(const phx_shard_t *s, uint64_t *step);
/* Host-blocking (waits for the last step's kernel, not for the device): clip coefficient and sum of squares
 * of the last step (1.0 / 0 if clip is off). */
PHX_API int phx_last_clip(phx_shard_t *s, float *coef, double *sumsq);
/* Number of kernels the library has launched on this handle (bench.py's gpu_launches). */
PHX_API int phx_kernel_launches(const phx_shard_t *s, uint64_t *count);
/* Snapshots that a later step superseded before the caller flushed them (see phx_step_and_snapshot's
 * contract), to the host replica and to the ring peers. */
PHX_API int phx_dropped_snapshots(const phx_shard_t *s, uint64_t *host, uint64_t *peers);
/* The derived AdamW scalars {decay, omb1, omb2, ss, sbc2} exactly as the library computes them: on the host
 * (binary64, individually rounded, works without a GPU) and by the device-side derivation of the
 * graph-capturable form for n step indices (host arrays in and out: out[5*i..]; host-blocking; needs a GPU).
 * Both must equal the oracle's bits; the tests pin them. */
PHX_API int phx_derived_scalars_host(float lr, float beta1, float beta2, float wd, uint64_t step, float out[5]);
PHX_API int phx_derived_scalars_device(float lr, float beta1, float beta2, float wd, const uint64_t *steps,
                                       uint32_t n, float *out);
PHX_API const char *phx_strerror(int err);
PHX_API int phx_last_cuda_error(const phx_shard_t *s);
PHX_API uint32_t phx_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PHX_H */
