// phx_api.cu — the C-ABI boundary (include/phx.h): shard definition, envelope, staging ring,
// chunked D2H flush with ping-pong host slots and DMA-ordered commit, restore.  Host logic only;
// every byte of the hot path is moved by the kernels in phx_kernels.cu or by the copy engines.
#include "../../include/phx.h"
#include "phx_kernels.cuh"

#include <cmath>
#include <cstring>
#include <new>
#include <vector>

namespace {

constexpr uint64_t kPadUnit = 64;      // elements; every rank's range is a multiple of 64
constexpr uint64_t kHeaderBytes = 256;
constexpr uint32_t kVersion = 1;
constexpr int kMaxDepth = 4;
#ifndef PHX_RESTORE_P2_CTAS
#define PHX_RESTORE_P2_CTAS 4
#endif
constexpr int kRestorePhase2Ctas = PHX_RESTORE_P2_CTAS;  // bulk-kernel CTAs of the second phase of phx_restore_async

struct Segment {
    uint32_t tensor_id;
    uint64_t off_in_tensor, off_in_shard, len;
    uint32_t flags;
};

enum SlotState { SLOT_EMPTY = 0, SLOT_INFLIGHT, SLOT_COMMITTED, SLOT_TORN_INFLIGHT, SLOT_TORN };

struct HostSlot {
    uint64_t step = 0;
    SlotState state = SLOT_EMPTY;
    phx_snapshot_header_t hdr{};  // the committed envelope this handle sent to the slot (valid while state != EMPTY)
};

// an event plus the capture sequence it was last recorded in (0 = recorded eagerly).  A wait is enqueued only
// when the waiting stream is in the same capture state: inside a capture the dependency on earlier eager work
// (or on an earlier replay) is already given by the launch stream's order, and an event recorded in a capture
// must not be waited on eagerly.
struct GraphEvent {
    cudaEvent_t ev = nullptr;
    unsigned long long cap = 0;
    bool valid = false;
};

// device scratch layout (bytes)
constexpr size_t kScrZeroHdr = 0;      // 256 zero bytes: invalidates a host slot header
constexpr size_t kScrOne = 256;        // float 1.0f: clip coefficient when clipping is off
constexpr size_t kScrCoef = 260;       // float: clip coefficient of the current step
constexpr size_t kScrSumsq = 264;      // double
constexpr size_t kScrHdr = 512;        // 2 x 256 B headers (direct mode)
constexpr size_t kScrHdrFull = kScrHdr + 2 * 256;  // kMaxDepth x 256 B full-rank-state headers (§8(f4))
constexpr size_t kScrBlock = kScrHdrFull + 4 * 256;  // phx::StepBlock of the graph-capturable form
constexpr size_t kScrBytes = kScrBlock + 1024;
static_assert(sizeof(phx::StepBlock) <= 1024, "step block must fit its scratch region");

uint64_t fnv1a64(const void *data, size_t len, uint64_t h = 0xCBF29CE484222325ull)
{
    const uint8_t *b = static_cast<const uint8_t *>(data);
    for (size_t i = 0; i < len; ++i) {
        h ^= b[i];
        h *= 0x100000001B3ull;
    }
    return h;
}

double pow_sqmul(double b, uint64_t t)  // LSB-first square-and-multiply, no libm pow
{
    double r = 1.0;
    while (t) {
        if (t & 1) r = r * b;
        b = b * b;
        t >>= 1;
    }
    return r;
}

inline bool aligned256(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 255u) == 0; }
inline bool aligned128(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 127u) == 0; }

}  // namespace

struct phx_shard {
    std::vector<phx_tensor_desc_t> layout;
    std::vector<Segment> segments;
    phx_config_t cfg{};
    phx_shard_info_t info{};
    // bound memory
    bool bound = false;
    float *d_p = nullptr, *d_m = nullptr, *d_v = nullptr;
    void *d_p16 = nullptr;
    uint8_t *d_staging = nullptr;
    uint8_t *h_replica = nullptr;
    uint8_t *d_replica = nullptr;  // device view of h_replica
    uint8_t *d_scratch = nullptr;
    double *d_partials = nullptr;  // 2 x sumsq_partials_count(n_padded): [a1 / phx_grad_sumsq_async | producer epilogue]
    int sm_count = 148;
    int device = -1;  // ordinal of the device that was current at phx_shard_bind; the hot calls check it
    // decay groups: class per 2048-element tile and the offsets where the flag toggles
    std::vector<uint8_t> decay_cls;
    std::vector<uint64_t> decay_bnd;
    uint32_t first_nodecay = 0;
    bool has_groups = false;
    uint8_t *d_decay = nullptr;  // device copy: toggles (8-byte aligned) then classes
    // state
    uint64_t last_step = 0;
    uint8_t user[128] = {0};
    uint32_t user_len = 0;
    uint8_t restored_user[128] = {0};
    uint32_t restored_user_len = 0;
    // staging ring / flush bookkeeping
    cudaEvent_t ev_step[kMaxDepth] = {nullptr, nullptr, nullptr, nullptr};
    cudaEvent_t ev_flush[kMaxDepth] = {nullptr, nullptr, nullptr, nullptr};
    bool flush_valid[kMaxDepth] = {false, false, false, false};
    cudaEvent_t ev_host[2] = {nullptr, nullptr};
    HostSlot host[2];
    int last_flush_slot = -1;  // staging slot whose ev_flush is the newest flush event
    int pending_slot = -1;     // staging slot holding a snapshot that has not been flushed
    uint64_t pending_step = 0;
    int64_t torn_chunks = -1;
    // §8(f1) peer replication: k device-addressable received buffers on the ring successors
    uint32_t n_peers = 0;
    uint8_t *d_peer[PHX_MAX_PEERS] = {nullptr, nullptr, nullptr, nullptr};
    cudaEvent_t ev_pflush[kMaxDepth] = {nullptr, nullptr, nullptr, nullptr};
    bool pflush_valid[kMaxDepth] = {false, false, false, false};
    cudaEvent_t ev_peer[2] = {nullptr, nullptr};
    HostSlot peer[2];              // bookkeeping of the peers' slot `step mod 2` (all k peers as one unit)
    int last_pflush_slot = -1;
    int pending_peer_slot = -1;
    uint64_t pending_peer_step = 0;
    int64_t torn_peer_chunks[PHX_MAX_PEERS] = {-1, -1, -1, -1};
    // k > 1: one library-owned copy stream per peer, forked from / joined into the caller's peer stream
    cudaStream_t peer_st[PHX_MAX_PEERS] = {nullptr, nullptr, nullptr, nullptr};
    cudaEvent_t ev_peer_fork = nullptr;
    cudaEvent_t ev_peer_join[PHX_MAX_PEERS] = {nullptr, nullptr, nullptr, nullptr};
    // §8(f3) publication of the model-param copy into other DP ranks' parameter buffers
    uint32_t n_pub = 0, pub_mode = PHX_PUBLISH_FUSED;
    uint8_t *d_pub[PHX_MAX_PARAM_PEERS] = {nullptr};
    cudaEvent_t ev_last_step = nullptr;  // recorded after every step's kernel (publication by copy engine waits on it)
    cudaEvent_t ev_pub = nullptr;        // the newest copy-engine publication has finished reading the model-param copy
    bool pub_valid = false;
    // §8(f4) full rank-state local snapshot: the model-parameter buffer W and its readiness / guard events
    uint8_t *d_W = nullptr;
    cudaEvent_t ev_params = nullptr;   // W holds every rank's parameters after step params_ready_step
    cudaEvent_t ev_wflush = nullptr;   // the newest local flush has finished reading W
    uint64_t params_ready_step = 0;
    bool params_ready = false, wflush_valid = false;
    // a6 in two phases (phx_restore_async): parameters (p, the model-param copy, W) in place / moments in place
    cudaEvent_t ev_rparams = nullptr, ev_rstate = nullptr;
    bool rparams_valid = false, rstate_valid = false;
    // misc
    int last_cuda_error = 0;
    uint64_t launches = 0;
    uint64_t dropped_host = 0, dropped_peers = 0;  // snapshots overwritten before they were flushed
    bool clip_valid = false;
    const double *clip_partials = nullptr;  // §8(e) global clip: one-shot per-rank sums for the next step
    uint32_t clip_count = 0;
    // graph-capturable form (include/phx.h "graph"): host mirror of the issue order; the device step block is the truth
    bool graph = false;
    uint64_t g_issue = 0;          // steps issued (captured or eager) since phx_graph_begin, on top of last_step at begin
    int g_pending_slot = -1;
    uint64_t g_pending_step = 0;
    int g_last_flush_slot = -1;
    int g_pending_peer_slot = -1;
    uint64_t g_pending_peer_step = 0;
    int g_last_pflush_slot = -1;
    GraphEvent gev_step[kMaxDepth], gev_flush[kMaxDepth], gev_pflush[kMaxDepth];
    GraphEvent gev_params, gev_wflush;  // §8(f4) in the graph form: W complete for g_params_step / newest flush done reading W
    uint64_t g_params_step = 0;
    bool g_params_ready = false;
};

#define PHX_CK(call)                                  \
    do {                                              \
        cudaError_t e__ = (call);                     \
        if (e__ != cudaSuccess) {                     \
            s->last_cuda_error = (int)e__;            \
            return PHX_ERR_CUDA;                      \
        }                                             \
    } while (0)

namespace {

void build_header(const phx_shard *s, uint64_t step, bool committed, phx_snapshot_header_t *h, uint32_t payload = 0)
{
    static_assert(sizeof(phx_snapshot_header_t) == 256, "envelope must be 256 bytes");
    std::memset(h, 0, sizeof(*h));
    std::memcpy(h->magic, "PHXSNAP1", 8);
    h->version = kVersion;
    h->header_bytes = (uint32_t)kHeaderBytes;
    h->seq_begin = step;
    h->step = step;
    h->n = s->info.n;
    h->n_padded = s->info.n_padded;
    h->total_numel = s->info.total_numel;
    h->shard_begin = s->info.shard_begin;
    h->layout_hash = s->info.layout_hash;
    h->dp_size = s->info.dp_size;
    h->dp_rank = s->info.dp_rank;
    h->tp_size = s->cfg.tp_size;
    h->tp_rank = s->cfg.tp_rank;
    h->pp_size = s->cfg.pp_size;
    h->pp_rank = s->cfg.pp_rank;
    h->chunk_bytes = s->cfg.chunk_bytes;
    h->user_len = s->user_len;
    h->payload = payload;
    std::memcpy(h->user, s->user, s->user_len);
    h->header_hash = fnv1a64(h, 240);
    h->seq_end = committed ? step : 0;
}

// commit rule: magic/version/size right, header hash matches, seq_begin == seq_end
bool header_valid(const phx_snapshot_header_t *h)
{
    if (std::memcmp(h->magic, "PHXSNAP1", 8) != 0) return false;
    if (h->version != kVersion || h->header_bytes != kHeaderBytes) return false;
    if (h->header_hash != fnv1a64(h, 240)) return false;
    return h->seq_begin == h->seq_end && h->seq_begin == h->step;
}

bool header_matches(const phx_shard *s, const phx_snapshot_header_t *h)
{
    return h->layout_hash == s->info.layout_hash && h->n == s->info.n && h->n_padded == s->info.n_padded &&
           h->total_numel == s->info.total_numel && h->shard_begin == s->info.shard_begin &&
           h->dp_size == s->info.dp_size && h->dp_rank == s->info.dp_rank && h->tp_size == s->cfg.tp_size &&
           h->tp_rank == s->cfg.tp_rank && h->pp_size == s->cfg.pp_size && h->pp_rank == s->cfg.pp_rank;
}

bool snapshots_on(const phx_shard *s) { return s->cfg.snapshot_disabled == 0; }
bool fp32_mode(const phx_shard *s) { return s->cfg.precision == PHX_PRECISION_FP32; }
uint32_t step_mode(const phx_shard *s)
{
    return (fp32_mode(s) ? (uint32_t)phx::kModeF32 : 0u) | (s->has_groups ? (uint32_t)phx::kModeGroups : 0u) |
           ((s->n_pub && s->pub_mode == PHX_PUBLISH_FUSED) ? (uint32_t)phx::kModePublish : 0u);
}
uint64_t model_elem_bytes(const phx_shard *s) { return fp32_mode(s) ? 4u : 2u; }
bool full_payload(const phx_shard *s) { return s->cfg.payload == PHX_PAYLOAD_FULL_RANK_STATE; }
uint32_t full_payload_word(const phx_shard *s) { return 1u | ((uint32_t)model_elem_bytes(s) << 8); }

// Decay groups: walk the rank's segments in shard order, record the offsets at which the no-decay flag
// toggles and classify every 2048-element tile as all-decay (0), all-no-decay (1) or mixed (2).  Pad
// lanes behind the last segment count as decayed (they hold zeros either way).
void build_decay_groups(phx_shard *s)
{
    const uint64_t L = s->info.n_padded;
    const uint64_t tile = 1ull << phx::kDecayTileShift;
    bool any = false;
    for (const auto &g : s->segments) any = any || (g.flags & PHX_TENSOR_NO_DECAY);
    s->has_groups = any;
    if (!any) return;
    s->first_nodecay = (!s->segments.empty() && s->segments[0].off_in_shard == 0 &&
                        (s->segments[0].flags & PHX_TENSOR_NO_DECAY)) ? 1u : 0u;
    uint32_t cur = s->first_nodecay;
    uint64_t pos = 0;
    auto toggle_to = [&](uint32_t f, uint64_t at) {
        if (f != cur && at < L) {
            s->decay_bnd.push_back(at);
            cur = f;
        }
    };
    for (const auto &g : s->segments) {
        if (g.len == 0) continue;
        toggle_to((g.flags & PHX_TENSOR_NO_DECAY) ? 1u : 0u, g.off_in_shard);
        pos = g.off_in_shard + g.len;
    }
    toggle_to(0u, pos);  // padding
    s->decay_cls.assign((size_t)((L + tile - 1) / tile), 0);
    size_t k = 0;        // toggles consumed so far
    uint32_t f = s->first_nodecay;
    for (size_t t = 0; t < s->decay_cls.size(); ++t) {
        const uint64_t lo = (uint64_t)t * tile, hi = lo + tile < L ? lo + tile : L;
        while (k < s->decay_bnd.size() && s->decay_bnd[k] <= lo) {
            f ^= 1u;
            ++k;
        }
        const bool mixed = k < s->decay_bnd.size() && s->decay_bnd[k] < hi;
        s->decay_cls[t] = mixed ? 2 : (uint8_t)f;
    }
}
bool direct_mode(const phx_shard *s) { return s->cfg.snapshot_source == PHX_SNAPSHOT_DIRECT; }
// SURVEY §8(b) "Ownership": a d_* pointer must be device (or managed) memory of the device the shard is bound on.
// A host pointer would be accepted by the launch and fault asynchronously, far from the call that caused it.
bool device_memory_on(const void *p, int dev)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    return (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged) && at.device == dev;
}

// The handle's events, scratch and function attributes belong to the device it was bound on; every later call
// assumes that device is current.  Checked in the hot calls (one thread-local read).
int check_device(phx_shard *s)
{
    int dev = -1;
    PHX_CK(cudaGetDevice(&dev));
    return dev == s->device ? PHX_OK : PHX_ERR_WRONG_DEVICE;
}

// number of ring positions the bookkeeping cycles through (direct mode: two header slots)
uint32_t ring_depth(const phx_shard *s) { return direct_mode(s) ? 2u : s->cfg.staging_depth; }

// settle the bookkeeping of host slots whose flush event has completed (block=true waits for it)
int settle_slots(phx_shard *s, HostSlot *slots, cudaEvent_t *evs, bool block)
{
    for (int i = 0; i < 2; ++i) {
        HostSlot &h = slots[i];
        if (h.state != SLOT_INFLIGHT && h.state != SLOT_TORN_INFLIGHT) continue;
        cudaError_t e = block ? cudaEventSynchronize(evs[i]) : cudaEventQuery(evs[i]);
        if (e == cudaErrorNotReady) continue;
        if (e != cudaSuccess) {
            s->last_cuda_error = (int)e;
            return PHX_ERR_CUDA;
        }
        h.state = h.state == SLOT_INFLIGHT ? SLOT_COMMITTED : SLOT_TORN;
    }
    return PHX_OK;
}
int settle_host_slots(phx_shard *s, bool block) { return settle_slots(s, s->host, s->ev_host, block); }
int settle_peer_slots(phx_shard *s, bool block) { return settle_slots(s, s->peer, s->ev_peer, block); }

// a4 + a5 for one destination slot (pinned host memory or a peer's received buffer): invalidate the
// destination header, copy the payload in chunk_bytes pieces (from the staging slot, or from the live
// planes in direct mode), copy the valid header last.  torn_chunks >= 0: stop after that many payload
// chunks and never commit (fault injection).
// full = true (§8(f4), local slot only): the model-parameter buffer W goes first, behind the optimizer part,
// and the committed header is the full-rank-state one; ev_wflush marks the end of the reads of W.
// graph-form events: a dependency edge inside a capture, a plain stream wait outside
unsigned long long capture_id(cudaStream_t st)
{
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    unsigned long long id = 0;
    if (cudaStreamGetCaptureInfo(st, &cs, &id) != cudaSuccess) {
        (void)cudaGetLastError();
        return 0;
    }
    return cs == cudaStreamCaptureStatusActive ? id : 0;
}
int gev_record(phx_shard *s, GraphEvent &g, cudaStream_t st)
{
    PHX_CK(cudaEventRecord(g.ev, st));
    g.cap = capture_id(st);
    g.valid = true;
    return PHX_OK;
}
int gev_wait(phx_shard *s, const GraphEvent &g, cudaStream_t st)
{
    if (g.valid && g.cap == capture_id(st)) PHX_CK(cudaStreamWaitEvent(st, g.ev, 0));
    return PHX_OK;
}

int enqueue_snapshot_copy(phx_shard *s, cudaStream_t st, uint8_t *dst, cudaMemcpyKind kind, int slot, int64_t torn_chunks,
                          bool full = false, GraphEvent *gev_w = nullptr)
{
    const bool direct = direct_mode(s);
    const uint8_t *src = direct ? nullptr : s->d_staging + (uint64_t)slot * s->info.slot_stride;
    const uint8_t *src_hdr = direct ? s->d_scratch + kScrHdr + (size_t)slot * kHeaderBytes : src;
    if (full) src_hdr = s->d_scratch + kScrHdrFull + (size_t)slot * kHeaderBytes;
    const bool torn = torn_chunks >= 0;
    // 1. invalidate the target slot's header; the OTHER slot keeps the previous committed snapshot
    PHX_CK(cudaMemcpyAsync(dst, s->d_scratch + kScrZeroHdr, kHeaderBytes, kind, st));
    // 2. payload in chunk_bytes pieces ("chunked")
    const uint64_t payload = s->info.snapshot_bytes - kHeaderBytes;
    const uint64_t chunk = s->cfg.chunk_bytes;
    uint64_t done_chunks = 0;
    bool stopped = false;
    if (full) {  // 2a. W, read from the live model-parameter buffer
        uint8_t *wdst = dst + s->info.snapshot_bytes;
        for (uint64_t off = 0; off < s->info.param_bytes; off += chunk, ++done_chunks) {
            if (torn && (int64_t)done_chunks >= torn_chunks) {
                stopped = true;
                break;
            }
            const uint64_t len = s->info.param_bytes - off < chunk ? s->info.param_bytes - off : chunk;
            PHX_CK(cudaMemcpyAsync(wdst + off, s->d_W + off, len, kind, st));
        }
        if (gev_w) {  // graph form: an edge of the captured graph, not the eager event
            const int rcw = gev_record(s, *gev_w, st);
            if (rcw != PHX_OK) return rcw;
        } else {
            PHX_CK(cudaEventRecord(s->ev_wflush, st));
            s->wflush_valid = true;
        }
    }
    for (uint64_t off = 0; off < payload && !stopped; off += chunk, ++done_chunks) {
        if (torn && (int64_t)done_chunks >= torn_chunks) break;
        const uint64_t len = payload - off < chunk ? payload - off : chunk;
        if (!direct) {
            PHX_CK(cudaMemcpyAsync(dst + kHeaderBytes + off, src + kHeaderBytes + off, len, kind, st));
        } else {
            // the chunk [off, off+len) of the packed payload p ‖ m ‖ v comes straight from the live planes;
            // a chunk that straddles a plane boundary is split there
            const uint64_t plane = 4 * s->info.n_padded;
            const uint8_t *planes[3] = {reinterpret_cast<const uint8_t *>(s->d_p), reinterpret_cast<const uint8_t *>(s->d_m),
                                        reinterpret_cast<const uint8_t *>(s->d_v)};
            uint64_t o = off, left = len;
            while (left) {
                const uint64_t pi = o / plane, po = o % plane;
                const uint64_t l = left < plane - po ? left : plane - po;
                PHX_CK(cudaMemcpyAsync(dst + kHeaderBytes + o, planes[pi] + po, l, kind, st));
                o += l;
                left -= l;
            }
        }
    }
    // 3. commit: the valid header (seq_end == seq_begin) lands last
    if (!torn) PHX_CK(cudaMemcpyAsync(dst, src_hdr, kHeaderBytes, kind, st));
    return PHX_OK;
}

}  // namespace

extern "C" {

uint32_t phx_version(void) { return 0x00010000u; }

const char *phx_strerror(int err)
{
    switch (err) {
    case PHX_OK: return "ok";
    case PHX_ERR_INVALID_ARG: return "invalid argument";
    case PHX_ERR_ALIGNMENT: return "pointer not 256-byte aligned";
    case PHX_ERR_NOT_BOUND: return "shard memory not bound";
    case PHX_ERR_STEP_ORDER: return "step is not last_step + 1";
    case PHX_ERR_NO_FLUSH_PENDING: return "no un-flushed snapshot";
    case PHX_ERR_NO_COMMITTED_SNAPSHOT: return "no committed snapshot in the replica";
    case PHX_ERR_LAYOUT_MISMATCH: return "replica belongs to a different logical shard";
    case PHX_ERR_CORRUPT_SLOT: return "replica slot is torn or corrupt";
    case PHX_ERR_CUDA: return "CUDA error (see phx_last_cuda_error)";
    case PHX_ERR_UNSUPPORTED_DEVICE: return "device is not compute capability 10.x";
    case PHX_ERR_SNAPSHOT_DISABLED: return "snapshots are disabled on this shard";
    case PHX_ERR_NOMEM: return "out of memory";
    case PHX_ERR_PARAMS_NOT_READY: return "model-parameter buffer not declared ready for this step";
    case PHX_ERR_GRAPH_MODE: return "call not available between phx_graph_begin and phx_graph_end (or outside them)";
    case PHX_ERR_WRONG_DEVICE: return "the current CUDA device is not the one the shard was bound on";
    case PHX_ERR_TOO_LARGE: return "more elements than the built-in scratch of the no-alloc entry point serves";
    default: return "unknown error";
    }
}

int phx_last_cuda_error(const phx_shard_t *s) { return s ? s->last_cuda_error : 0; }

// ---- a0 -------------------------------------------------------------------------------------
int phx_shard_create(const phx_tensor_desc_t *layout, size_t n_tensors, uint32_t dp_size, uint32_t dp_rank,
                     const phx_config_t *cfg, phx_shard_t **out)
{
    if (!out) return PHX_ERR_INVALID_ARG;
    *out = nullptr;
    if ((!layout && n_tensors) || dp_size == 0 || dp_rank >= dp_size) return PHX_ERR_INVALID_ARG;
    phx_shard *s = new (std::nothrow) phx_shard();
    if (!s) return PHX_ERR_NOMEM;
    if (cfg) s->cfg = *cfg;
    phx_config_t &c = s->cfg;
    if (c.tp_size == 0) c.tp_size = 1;
    if (c.pp_size == 0) c.pp_size = 1;
    if (c.staging_depth == 0) c.staging_depth = 2;
    if (c.chunk_bytes == 0) c.chunk_bytes = 32ull << 20;
    c.chunk_bytes = (c.chunk_bytes + 255) & ~255ull;
    if (c.tp_rank >= c.tp_size || c.pp_rank >= c.pp_size || c.staging_depth > kMaxDepth ||
        c.sync_mode > PHX_SYNC_RELAXED || c.restore_mode > PHX_RESTORE_BULK_KERNEL || !(c.max_grad_norm == c.max_grad_norm) ||
        c.snapshot_source > PHX_SNAPSHOT_DIRECT || c.precision > PHX_PRECISION_FP32 ||
        c.payload > PHX_PAYLOAD_FULL_RANK_STATE || (c.payload == PHX_PAYLOAD_FULL_RANK_STATE && c.snapshot_disabled) ||
        (c.snapshot_source == PHX_SNAPSHOT_DIRECT && c.sync_mode != PHX_SYNC_STRICT)) {
        delete s;
        return PHX_ERR_INVALID_ARG;
    }
    s->layout.assign(layout, layout + n_tensors);

    uint64_t total = 0;
    for (const auto &t : s->layout) total += t.numel;
    const uint64_t unit = kPadUnit * dp_size;
    const uint64_t L = ((total + unit - 1) / unit) * kPadUnit;
    const uint64_t begin = (uint64_t)dp_rank * L, end = begin + L;
    uint64_t n = total > begin ? total - begin : 0;
    if (n > L) n = L;

    uint64_t t0 = 0;
    for (const auto &t : s->layout) {
        const uint64_t t1 = t0 + t.numel;
        const uint64_t lo = t0 > begin ? t0 : begin, hi = t1 < end ? t1 : end;
        if (hi > lo) s->segments.push_back(Segment{t.tensor_id, lo - t0, lo - begin, hi - lo, t.flags});
        t0 = t1;
    }
    // layout hash: per tensor (numel u64, tensor_id u32, flags u32), then dp_size, tp_size, tp_rank, pp_size, pp_rank
    uint64_t h = 0xCBF29CE484222325ull;
    for (const auto &t : s->layout) {
        uint8_t rec[16];
        std::memcpy(rec, &t.numel, 8);
        std::memcpy(rec + 8, &t.tensor_id, 4);
        std::memcpy(rec + 12, &t.flags, 4);
        h = fnv1a64(rec, 16, h);
    }
    const uint32_t coords[5] = {dp_size, c.tp_size, c.tp_rank, c.pp_size, c.pp_rank};
    h = fnv1a64(coords, sizeof(coords), h);

    phx_shard_info_t &i = s->info;
    i.n = n;
    i.n_padded = L;
    i.total_numel = total;
    i.shard_begin = begin;
    i.layout_hash = h;
    i.snapshot_bytes = kHeaderBytes + 12 * L;
    i.slot_stride = (i.snapshot_bytes + 255) & ~255ull;
    i.n_segments = (uint32_t)s->segments.size();
    i.staging_depth = c.snapshot_source == PHX_SNAPSHOT_DIRECT ? 0 : c.staging_depth;
    i.dp_size = dp_size;
    i.dp_rank = dp_rank;
    i.param_bytes = (uint64_t)dp_size * L * model_elem_bytes(s);
    i.host_snapshot_bytes = i.snapshot_bytes + (full_payload(s) ? i.param_bytes : 0);
    i.host_slot_stride = (i.host_snapshot_bytes + 255) & ~255ull;
    build_decay_groups(s);
    *out = s;
    return PHX_OK;
}

int phx_shard_destroy(phx_shard_t *s)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (s->bound) {
        settle_host_slots(s, true);
        for (int k = 0; k < kMaxDepth; ++k) {
            if (s->ev_step[k]) cudaEventSynchronize(s->ev_step[k]), cudaEventDestroy(s->ev_step[k]);
            if (s->ev_flush[k]) cudaEventSynchronize(s->ev_flush[k]), cudaEventDestroy(s->ev_flush[k]);
        }
        settle_peer_slots(s, true);
        for (int k = 0; k < kMaxDepth; ++k)
            if (s->ev_pflush[k]) cudaEventSynchronize(s->ev_pflush[k]), cudaEventDestroy(s->ev_pflush[k]);
        for (int k = 0; k < 2; ++k) {
            if (s->ev_host[k]) cudaEventDestroy(s->ev_host[k]);
            if (s->ev_peer[k]) cudaEventDestroy(s->ev_peer[k]);
        }
        if (s->ev_last_step) cudaEventSynchronize(s->ev_last_step), cudaEventDestroy(s->ev_last_step);
        if (s->ev_pub) cudaEventSynchronize(s->ev_pub), cudaEventDestroy(s->ev_pub);
        if (s->ev_peer_fork) cudaEventDestroy(s->ev_peer_fork);
        for (int k = 0; k < PHX_MAX_PEERS; ++k) {
            if (s->ev_peer_join[k]) cudaEventDestroy(s->ev_peer_join[k]);
            if (s->peer_st[k]) cudaStreamSynchronize(s->peer_st[k]), cudaStreamDestroy(s->peer_st[k]);
        }
        for (int k = 0; k < kMaxDepth; ++k) {
            if (s->gev_step[k].ev) cudaEventDestroy(s->gev_step[k].ev);
            if (s->gev_flush[k].ev) cudaEventDestroy(s->gev_flush[k].ev);
            if (s->gev_pflush[k].ev) cudaEventDestroy(s->gev_pflush[k].ev);
        }
        if (s->gev_params.ev) cudaEventDestroy(s->gev_params.ev);
        if (s->gev_wflush.ev) cudaEventDestroy(s->gev_wflush.ev);
        if (s->ev_rparams) cudaEventDestroy(s->ev_rparams);
        if (s->ev_rstate) cudaEventSynchronize(s->ev_rstate), cudaEventDestroy(s->ev_rstate);
        if (s->ev_params) cudaEventDestroy(s->ev_params);
        if (s->ev_wflush) cudaEventDestroy(s->ev_wflush);
        if (s->d_scratch) cudaFree(s->d_scratch);
        if (s->d_partials) cudaFree(s->d_partials);
        if (s->d_decay) cudaFree(s->d_decay);
    }
    delete s;
    return PHX_OK;
}

int phx_shard_info(const phx_shard_t *s, phx_shard_info_t *out)
{
    if (!s || !out) return PHX_ERR_INVALID_ARG;
    *out = s->info;
    return PHX_OK;
}

int phx_shard_segments(const phx_shard_t *s, uint32_t *tensor_id, uint64_t *off_in_tensor, uint64_t *off_in_shard,
                       uint64_t *len, uint32_t cap)
{
    if (!s || (cap && (!tensor_id || !off_in_tensor || !off_in_shard || !len))) return PHX_ERR_INVALID_ARG;
    for (uint32_t k = 0; k < cap && k < s->segments.size(); ++k) {
        tensor_id[k] = s->segments[k].tensor_id;
        off_in_tensor[k] = s->segments[k].off_in_tensor;
        off_in_shard[k] = s->segments[k].off_in_shard;
        len[k] = s->segments[k].len;
    }
    return PHX_OK;
}

// ---- binding ----------------------------------------------------------------------------------
int phx_shard_bind(phx_shard_t *s, float *d_p, float *d_m, float *d_v, void *d_p_bf16, void *d_staging,
                   void *h_replica)
{
    if (!s || !d_p || !d_m || !d_v || (!d_p_bf16 && !fp32_mode(s))) return PHX_ERR_INVALID_ARG;
    if (snapshots_on(s) && !d_staging && !direct_mode(s)) return PHX_ERR_INVALID_ARG;
    // d_p_bf16 may be the rank's range inside its model-parameter buffer (§8(f3)): r * n_padded * 2 bytes, a multiple of 128
    if (!aligned256(d_p) || !aligned256(d_m) || !aligned256(d_v) || !aligned128(d_p_bf16) || !aligned256(d_staging) ||
        !aligned256(h_replica))
        return PHX_ERR_ALIGNMENT;
    if (s->bound) return PHX_ERR_INVALID_ARG;

    int dev = 0, major = 0;
    PHX_CK(cudaGetDevice(&dev));
    PHX_CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return PHX_ERR_UNSUPPORTED_DEVICE;  // sm_100a only; deliberately no fallback
    PHX_CK(cudaDeviceGetAttribute(&s->sm_count, cudaDevAttrMultiProcessorCount, dev));
    for (const void *p : {static_cast<const void *>(d_p), static_cast<const void *>(d_m), static_cast<const void *>(d_v),
                          static_cast<const void *>(d_p_bf16), static_cast<const void *>(d_staging)})
        if (p != nullptr && !device_memory_on(p, dev)) return PHX_ERR_INVALID_ARG;
    s->device = dev;

    if (snapshots_on(s) && h_replica) {
        void *dview = nullptr;
        cudaError_t e = cudaHostGetDevicePointer(&dview, h_replica, 0);
        if (e != cudaSuccess) {  // not pinned/mapped host memory
            s->last_cuda_error = (int)e;
            (void)cudaGetLastError();
            return PHX_ERR_INVALID_ARG;
        }
        s->d_replica = static_cast<uint8_t *>(dview);
    }
    PHX_CK(cudaMalloc(reinterpret_cast<void **>(&s->d_scratch), kScrBytes));
    PHX_CK(cudaMemset(s->d_scratch, 0, kScrBytes));
    PHX_CK(cudaMalloc(reinterpret_cast<void **>(&s->d_partials), 2 * phx::sumsq_partials_count(s->info.n_padded) * sizeof(double)));
    const float one = 1.0f;
    PHX_CK(cudaMemcpy(s->d_scratch + kScrOne, &one, 4, cudaMemcpyHostToDevice));
    PHX_CK(cudaMemcpy(s->d_scratch + kScrCoef, &one, 4, cudaMemcpyHostToDevice));
    for (uint32_t k = 0; k < ring_depth(s); ++k) {
        PHX_CK(cudaEventCreateWithFlags(&s->ev_step[k], cudaEventDisableTiming));
        PHX_CK(cudaEventCreateWithFlags(&s->ev_flush[k], cudaEventDisableTiming));
        PHX_CK(cudaEventCreateWithFlags(&s->ev_pflush[k], cudaEventDisableTiming));
    }
    PHX_CK(cudaEventCreateWithFlags(&s->ev_last_step, cudaEventDisableTiming));
    PHX_CK(cudaEventCreateWithFlags(&s->ev_pub, cudaEventDisableTiming));
    for (int k = 0; k < kMaxDepth; ++k) {
        PHX_CK(cudaEventCreateWithFlags(&s->gev_step[k].ev, cudaEventDisableTiming));
        PHX_CK(cudaEventCreateWithFlags(&s->gev_flush[k].ev, cudaEventDisableTiming));
        PHX_CK(cudaEventCreateWithFlags(&s->gev_pflush[k].ev, cudaEventDisableTiming));
    }
    PHX_CK(cudaEventCreateWithFlags(&s->gev_params.ev, cudaEventDisableTiming));
    PHX_CK(cudaEventCreateWithFlags(&s->gev_wflush.ev, cudaEventDisableTiming));
    PHX_CK(cudaEventCreateWithFlags(&s->ev_rparams, cudaEventDisableTiming));
    PHX_CK(cudaEventCreateWithFlags(&s->ev_rstate, cudaEventDisableTiming));
    PHX_CK(cudaEventCreateWithFlags(&s->ev_params, cudaEventDisableTiming));
    PHX_CK(cudaEventCreateWithFlags(&s->ev_wflush, cudaEventDisableTiming));
    for (int k = 0; k < 2; ++k) {
        PHX_CK(cudaEventCreateWithFlags(&s->ev_host[k], cudaEventDisableTiming));
        PHX_CK(cudaEventCreateWithFlags(&s->ev_peer[k], cudaEventDisableTiming));
    }
    if (s->has_groups) {
        const size_t nb = s->decay_bnd.size() * sizeof(uint64_t);
        PHX_CK(cudaMalloc(reinterpret_cast<void **>(&s->d_decay), nb + s->decay_cls.size() + 8));
        if (nb) PHX_CK(cudaMemcpy(s->d_decay, s->decay_bnd.data(), nb, cudaMemcpyHostToDevice));
        PHX_CK(cudaMemcpy(s->d_decay + nb, s->decay_cls.data(), s->decay_cls.size(), cudaMemcpyHostToDevice));
    }

    s->d_p = d_p;
    s->d_m = d_m;
    s->d_v = d_v;
    s->d_p16 = d_p_bf16;
    s->d_staging = static_cast<uint8_t *>(d_staging);
    s->h_replica = static_cast<uint8_t *>(h_replica);
    s->bound = true;
    return PHX_OK;
}

int phx_shard_set_state(phx_shard_t *s, uint64_t step, void *stream)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    if (!fp32_mode(s)) {
        PHX_CK(phx::launch_regen_bf16(s->d_p, s->d_p16, s->info.n_padded, static_cast<cudaStream_t>(stream)));
        s->launches += s->info.n_padded ? 1 : 0;
    }
    s->last_step = step;
    s->pending_slot = -1;
    s->pending_peer_slot = -1;
    return PHX_OK;
}

int phx_set_user_metadata(phx_shard_t *s, const void *blob, uint32_t len)
{
    if (!s || len > 128 || (len && !blob)) return PHX_ERR_INVALID_ARG;
    // the graph form keeps the envelope template on the device: phx_graph_set_user_metadata updates it in stream order
    if (s->graph) return PHX_ERR_GRAPH_MODE;
    std::memset(s->user, 0, sizeof(s->user));
    if (len) std::memcpy(s->user, blob, len);
    s->user_len = len;
    return PHX_OK;
}

// ---- a1 + a2 + a3 --------------------------------------------------------------------------------
namespace {

// derived scalars: double on the host, every operation individually rounded (the file is compiled with
// -ffp-contract=off), rounded once to fp32 (include/phx.h a3, reading R6)
void derive_scalars_host(float lr, float beta1, float beta2, float eps, float wd, uint64_t step, phx::AdamScalars *sc)
{
    const double dlr = lr, db1 = beta1, db2 = beta2, dwd = wd;
    sc->beta1 = beta1;
    sc->beta2 = beta2;
    sc->eps = eps;
    const double lw = dlr * dwd;
    sc->decay = (float)(1.0 - lw);
    sc->omb1 = (float)(1.0 - db1);
    sc->omb2 = (float)(1.0 - db2);
    const double b1t = pow_sqmul(db1, step), b2t = pow_sqmul(db2, step);
    sc->ss = (float)(dlr / (1.0 - b1t));
    sc->sbc2 = (float)std::sqrt(1.0 - b2t);
}

// a1: optional clip — from the one-shot partials the caller exchanged (§8(e), §8(f4b)) or by the shard's own pass
int enqueue_clip(phx_shard *s, const void *d_grads, phx::StepArgs &a, cudaStream_t st)
{
    a.coef = reinterpret_cast<const float *>(s->d_scratch + kScrOne);
    s->clip_valid = false;
    if (!(s->cfg.max_grad_norm > 0.0f)) return PHX_OK;
    if (s->clip_partials != nullptr) {
        PHX_CK(phx::launch_clip_from_partials(s->clip_partials, s->clip_count, s->cfg.max_grad_norm,
                                              reinterpret_cast<double *>(s->d_scratch + kScrSumsq),
                                              reinterpret_cast<float *>(s->d_scratch + kScrCoef), st));
        s->launches += 1;
        s->clip_partials = nullptr;
        s->clip_count = 0;
    } else {
        int nl = 0;
        PHX_CK(phx::launch_sumsq_clip(d_grads, fp32_mode(s), s->info.n_padded, s->cfg.max_grad_norm, s->d_partials,
                                      reinterpret_cast<double *>(s->d_scratch + kScrSumsq),
                                      reinterpret_cast<float *>(s->d_scratch + kScrCoef), st, &nl));
        s->launches += nl;
    }
    a.coef = reinterpret_cast<const float *>(s->d_scratch + kScrCoef);
    s->clip_valid = true;
    return PHX_OK;
}

void fill_common_args(const phx_shard *s, const void *d_grads, int slot, phx::StepArgs &a)
{
    if (slot >= 0) {
        if (direct_mode(s)) {
            a.shdr = s->d_scratch + kScrHdr + (size_t)slot * kHeaderBytes;  // header only; planes stay live
        } else {
            uint8_t *base = s->d_staging + (uint64_t)slot * s->info.slot_stride;
            a.shdr = base;
            a.sp = reinterpret_cast<float *>(base + kHeaderBytes);
            a.sm = a.sp + s->info.n_padded;
            a.sv = a.sm + s->info.n_padded;
        }
    }
    a.p = s->d_p;
    a.m = s->d_m;
    a.v = s->d_v;
    a.g = d_grads;
    a.p16 = s->d_p16;
    a.n_padded = s->info.n_padded;
    if (s->has_groups) {
        a.decay_bnd = reinterpret_cast<const uint64_t *>(s->d_decay);
        a.decay_cls = s->d_decay + s->decay_bnd.size() * sizeof(uint64_t);
        a.n_bnd = (uint32_t)s->decay_bnd.size();
        a.first_nodecay = s->first_nodecay;
    }
    if (s->n_pub && s->pub_mode == PHX_PUBLISH_FUSED) {
        a.n_pub = s->n_pub;
        for (uint32_t q = 0; q < s->n_pub; ++q)
            a.pub[q] = s->d_pub[q] + (uint64_t)s->info.dp_rank * s->info.n_padded * model_elem_bytes(s);
    }
}

}  // namespace

int phx_step_and_snapshot(phx_shard_t *s, const void *d_grads, float lr, float beta1, float beta2, float eps,
                          float wd, uint64_t step, void *stream)
{
    if (!s || !d_grads) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    if (s->graph) return PHX_ERR_GRAPH_MODE;
    if (int rcd = check_device(s)) return rcd;
    if (!aligned256(d_grads)) return PHX_ERR_ALIGNMENT;
    if (step != s->last_step + 1) return PHX_ERR_STEP_ORDER;  // I4 step atomicity
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const bool snap = snapshots_on(s);

    phx::StepArgs a;
    std::memset(&a, 0, sizeof(a));
    derive_scalars_host(lr, beta1, beta2, eps, wd, step, &a.sc);
    int rc = enqueue_clip(s, d_grads, a, st);
    if (rc != PHX_OK) return rc;

    int slot = -1;
    if (snap) {
        slot = (int)(step % ring_depth(s));
        // a2: the single sync point — stream-side wait, the host never blocks
        // ("guarantees the peer-resident replica is fully committed before the optimizer mutates the protected state")
        if (s->cfg.sync_mode == PHX_SYNC_STRICT) {
            if (s->last_flush_slot >= 0) PHX_CK(cudaStreamWaitEvent(st, s->ev_flush[s->last_flush_slot], 0));
            if (s->last_pflush_slot >= 0) PHX_CK(cudaStreamWaitEvent(st, s->ev_pflush[s->last_pflush_slot], 0));
        } else {
            if (s->flush_valid[slot]) PHX_CK(cudaStreamWaitEvent(st, s->ev_flush[slot], 0));
            if (s->pflush_valid[slot]) PHX_CK(cudaStreamWaitEvent(st, s->ev_pflush[slot], 0));
            // §8(f4): the full-rank-state flush reads the live W (this rank's range of it is d_p_bf16) whatever the
            // staging depth, so even a relaxed step must not start before the newest flush has finished READING W
            if (full_payload(s) && s->wflush_valid) PHX_CK(cudaStreamWaitEvent(st, s->ev_wflush, 0));
        }
        // contract: a snapshot the caller never flushed is overwritten by its successor's slot reuse / superseded;
        // it is counted, not an error (phx_dropped_snapshots)
        if (s->pending_slot >= 0 && s->h_replica) s->dropped_host += 1;
        if (s->pending_peer_slot >= 0 && s->n_peers) s->dropped_peers += 1;
        phx_snapshot_header_t hdr;
        build_header(s, step, true, &hdr);
        std::memcpy(&a.hdr, &hdr, sizeof(hdr));
        if (full_payload(s)) {  // §8(f4): the local slot's envelope differs in the payload word and the hash
            phx_snapshot_header_t hf;
            build_header(s, step, true, &hf, full_payload_word(s));
            a.shdr_full = s->d_scratch + kScrHdrFull + (size_t)slot * kHeaderBytes;
            a.full_payload = hf.payload;
            a.full_hash = hf.header_hash;
        }
    }
    // a copy-engine publication of the previous step may still be reading the model-param copy this kernel rewrites
    if (s->pub_valid) PHX_CK(cudaStreamWaitEvent(st, s->ev_pub, 0));
    fill_common_args(s, d_grads, slot, a);

    // a two-phase restore (phx_restore_async) may still be bringing m and v back on its side stream
    if (s->rstate_valid) {
        PHX_CK(cudaStreamWaitEvent(st, s->ev_rstate, 0));
        s->rstate_valid = false;  // later steps follow this one in the caller's stream order
    }
    // a3: one kernel, one pass
    PHX_CK(phx::launch_step(a, snap && !direct_mode(s), step_mode(s), false, st));
    s->launches += s->info.n_padded ? 1 : 0;
    PHX_CK(cudaEventRecord(s->ev_last_step, st));
    if (snap) {
        PHX_CK(cudaEventRecord(s->ev_step[slot], st));
        s->pending_slot = slot;
        s->pending_step = step;
        s->pending_peer_slot = slot;
        s->pending_peer_step = step;
    }
    s->last_step = step;
    s->params_ready = false;
    return PHX_OK;
}

// ---- a4 + a5 -------------------------------------------------------------------------------------
int phx_snapshot_flush_async(phx_shard_t *s, void *side_stream)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound || (snapshots_on(s) && !s->h_replica)) return PHX_ERR_NOT_BOUND;
    if (!snapshots_on(s)) return PHX_ERR_SNAPSHOT_DISABLED;
    if (s->graph) return PHX_ERR_GRAPH_MODE;
    if (int rcd = check_device(s)) return rcd;
    if (s->pending_slot < 0) return PHX_ERR_NO_FLUSH_PENDING;
    cudaStream_t st = static_cast<cudaStream_t>(side_stream);
    const int slot = s->pending_slot;
    const uint64_t step = s->pending_step;
    const int hs = (int)(step & 1);  // ping-pong
    uint8_t *dst = s->h_replica + (uint64_t)hs * s->info.host_slot_stride;
    const bool full = full_payload(s);
    if (full) {
        if (!s->d_W) return PHX_ERR_NOT_BOUND;
        if (!s->params_ready || s->params_ready_step != step) return PHX_ERR_PARAMS_NOT_READY;
        PHX_CK(cudaStreamWaitEvent(st, s->ev_params, 0));  // the all-gather of this step has landed in W
    }

    PHX_CK(cudaStreamWaitEvent(st, s->ev_step[slot], 0));  // the step's kernel has written the slot
    if (s->last_flush_slot >= 0)                            // flushes are serialised whatever stream they use
        PHX_CK(cudaStreamWaitEvent(st, s->ev_flush[s->last_flush_slot], 0));

    const bool torn = s->torn_chunks >= 0;
    s->host[hs].step = step;
    s->host[hs].state = torn ? SLOT_TORN_INFLIGHT : SLOT_INFLIGHT;
    build_header(s, step, true, &s->host[hs].hdr, full ? full_payload_word(s) : 0u);  // what lands last, if it lands
    int rc = enqueue_snapshot_copy(s, st, dst, cudaMemcpyDeviceToHost, slot, s->torn_chunks, full);
    if (rc != PHX_OK) return rc;
    PHX_CK(cudaEventRecord(s->ev_flush[slot], st));
    PHX_CK(cudaEventRecord(s->ev_host[hs], st));
    s->flush_valid[slot] = true;
    s->last_flush_slot = slot;
    s->pending_slot = -1;
    s->torn_chunks = -1;
    return PHX_OK;
}

int phx_snapshot_wait(phx_shard_t *s, uint64_t step)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    const int hs = (int)(step & 1);
    if (s->host[hs].state == SLOT_EMPTY || s->host[hs].step != step) return PHX_ERR_NO_COMMITTED_SNAPSHOT;
    int rc = settle_host_slots(s, true);
    if (rc != PHX_OK) return rc;
    return s->host[hs].state == SLOT_COMMITTED ? PHX_OK : PHX_ERR_CORRUPT_SLOT;
}

int phx_snapshot_query(phx_shard_t *s, uint64_t *newest_committed_step, int *slot)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    int rc = settle_host_slots(s, false);
    if (rc != PHX_OK) return rc;
    int best = -1;
    for (int i = 0; i < 2; ++i)
        if (s->host[i].state == SLOT_COMMITTED && (best < 0 || s->host[i].step > s->host[best].step)) best = i;
    if (best < 0) return PHX_ERR_NO_COMMITTED_SNAPSHOT;
    if (newest_committed_step) *newest_committed_step = s->host[best].step;
    if (slot) *slot = best;
    return PHX_OK;
}

int phx_fault_inject_torn_flush(phx_shard_t *s, int64_t payload_chunks)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    s->torn_chunks = payload_chunks < 0 ? -1 : payload_chunks;
    return PHX_OK;
}

// ---- a6 ------------------------------------------------------------------------------------------
namespace {

// Choose between two envelopes the valid, identity-matching one with the largest step.
int choose_slot(const phx_shard *s, const phx_snapshot_header_t hdr[2], const bool usable[2], uint32_t want_payload,
                bool ok[2])
{
    int best = -1;
    bool any_valid = false;
    for (int i = 0; i < 2; ++i) {
        ok[i] = false;
        if (!usable[i] || !header_valid(&hdr[i])) continue;
        any_valid = true;
        if (!header_matches(s, &hdr[i]) || hdr[i].payload != want_payload) continue;
        ok[i] = true;
        if (best < 0 || hdr[i].step > hdr[best].step) best = i;
    }
    if (best < 0) return any_valid ? PHX_ERR_LAYOUT_MISMATCH : PHX_ERR_NO_COMMITTED_SNAPSHOT;
    return best;
}

// Enqueue the rebuild of the live shard from slot `best` of a replica (two slots `stride` apart).
// copy_src: address for copy-engine copies; kern_src: device-visible address for the bulk kernel.
// two_phase (phx_restore_async, reading R37): p -> model-param copy [-> W] -> ev_rparams -> m, v -> ev_rstate
// on the one stream `st`; the recomputed iteration's forward/backward may start at ev_rparams, the next optimizer
// step waits for ev_rstate by itself.
int enqueue_restore(phx_shard *s, int best, const phx_snapshot_header_t &hdr, const uint8_t *copy_src,
                    const uint8_t *kern_src, cudaStream_t st, uint64_t stride, uint32_t want_payload, bool two_phase = false)
{
    // The copies overwrite the live planes (and W): order them behind everything of THIS handle that may still be
    // reading or writing them — the newest step's kernel, a direct-source flush to the host or to the peers, a
    // full-rank-state flush reading W, a copy-engine publication, an earlier two-phase restore.
    if (s->last_step > 0 || s->ev_last_step) PHX_CK(cudaStreamWaitEvent(st, s->ev_last_step, 0));
    if (s->last_flush_slot >= 0) PHX_CK(cudaStreamWaitEvent(st, s->ev_flush[s->last_flush_slot], 0));
    if (s->last_pflush_slot >= 0) PHX_CK(cudaStreamWaitEvent(st, s->ev_pflush[s->last_pflush_slot], 0));
    if (s->wflush_valid) PHX_CK(cudaStreamWaitEvent(st, s->ev_wflush, 0));
    if (s->pub_valid) PHX_CK(cudaStreamWaitEvent(st, s->ev_pub, 0));
    if (s->rstate_valid) PHX_CK(cudaStreamWaitEvent(st, s->ev_rstate, 0));
    s->rparams_valid = s->rstate_valid = false;

    const uint64_t N = s->info.n_padded;
    const uint64_t off = (uint64_t)best * stride + kHeaderBytes;
    const bool bulk = s->cfg.restore_mode == PHX_RESTORE_BULK_KERNEL;
    void *p16 = fp32_mode(s) ? nullptr : s->d_p16;
    const float *ksrc = reinterpret_cast<const float *>(kern_src + off);
    const uint8_t *src = copy_src + off;
    // planes [first, first + count) of p ‖ m ‖ v -> the live planes; with_p16: regenerate the model-param copy from p
    auto planes = [&](int first, int count, bool with_p16, int ctas) -> int {
        float *dst[3] = {s->d_p, s->d_m, s->d_v};
        if (bulk) {
            phx::RestorePlanes pl{{nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr}, count};
            for (int k = 0; k < count; ++k) {
                pl.src[k] = ksrc + (uint64_t)(first + k) * N;
                pl.dst[k] = dst[first + k];
            }
            PHX_CK(phx::launch_restore_bulk(pl, with_p16 ? p16 : nullptr, N, ctas, st));
            s->launches += N ? 1 : 0;
        } else {
            for (int k = first; k < first + count; ++k)
                PHX_CK(cudaMemcpyAsync(dst[k], src + (uint64_t)k * 4 * N, 4 * N, cudaMemcpyDefault, st));
            if (with_p16 && p16) {
                PHX_CK(phx::launch_regen_bf16(s->d_p, s->d_p16, N, st));
                s->launches += N ? 1 : 0;
            }
        }
        return PHX_OK;
    };
    const uint8_t *wsrc = copy_src + off + 12 * N;  // §8(f4): W sits behind the optimizer part of the same slot
    int rc = PHX_OK;
    if (!two_phase) {
        if ((rc = planes(0, 3, true, 2 * s->sm_count)) != PHX_OK) return rc;
        if (want_payload != 0)  // in-place recovery: W comes back from the same slot, no other rank is read
            PHX_CK(cudaMemcpyAsync(s->d_W, wsrc, s->info.param_bytes, cudaMemcpyDefault, st));
    } else {
        // phase 1 = what the recomputed iteration's forward/backward reads.  Optimizer-only payload: p, from which the
        // model-param copy is regenerated.  Full rank state: W ALONE — the rank's own range of it (d_p_bf16, enforced
        // by phx_shard_bind_params) is part of the snapshot's W, so p can wait for phase 2 with the moments.
        if (want_payload != 0) {
            PHX_CK(cudaMemcpyAsync(s->d_W, wsrc, s->info.param_bytes, cudaMemcpyDefault, st));
        } else if ((rc = planes(0, 1, true, 2 * s->sm_count)) != PHX_OK) {
            return rc;
        }
        PHX_CK(cudaEventRecord(s->ev_rparams, st));
        s->rparams_valid = true;
        // phase 2 runs BESIDE the recomputed iteration's kernels: FOUR persistent CTAs of the bulk kernel already
        // saturate the host link (2: 86 %; 8-37: the same rate, but each CTA's 96 KB of shared memory takes an SM away
        // from the forward/backward — profiles/r02c_restore_bulk.md), the other 144 SMs stay with the compute
        rc = want_payload != 0 ? planes(0, 3, false, kRestorePhase2Ctas) : planes(1, 2, false, kRestorePhase2Ctas);
        if (rc != PHX_OK) return rc;
        PHX_CK(cudaEventRecord(s->ev_rstate, st));
        s->rstate_valid = true;
    }
    PHX_CK(cudaEventRecord(s->ev_last_step, st));  // later flushes / publications order behind the restore
    s->last_step = hdr.step;
    s->pending_slot = -1;
    s->pending_peer_slot = -1;
    s->params_ready = false;
    s->clip_partials = nullptr;  // the recompute of the in-flight step exchanges its sums again
    s->clip_count = 0;
    s->restored_user_len = hdr.user_len <= 128 ? hdr.user_len : 128;
    std::memcpy(s->restored_user, hdr.user, 128);
    return PHX_OK;
}

}  // namespace

// Enqueue-only: the host never waits for the device here.  Which slot to take is decided from
//   - the envelope IN the pinned host slot, read with a plain memcpy, for a slot this handle is not writing
//     (never used by this handle, or its flush event has completed — cudaEventQuery, non-blocking);
//   - the handle's own commit bookkeeping for a slot whose flush is still in flight: the envelope it sent is
//     known, the flush cannot tear (a torn flush is known as such and skipped), and `stream` is made to wait
//     for the flush event before the copies, so the payload has landed when it is read.
namespace {
int restore_own(phx_shard *s, void *stream, uint64_t *restored_step, bool two_phase)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound || (snapshots_on(s) && !s->h_replica)) return PHX_ERR_NOT_BOUND;
    if (!snapshots_on(s)) return PHX_ERR_SNAPSHOT_DISABLED;
    if (s->graph) return PHX_ERR_GRAPH_MODE;
    if (full_payload(s) && !s->d_W) return PHX_ERR_NOT_BOUND;
    if (int rcd = check_device(s)) return rcd;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int rc = settle_host_slots(s, false);
    if (rc != PHX_OK) return rc;
    phx_snapshot_header_t hdr[2];
    bool usable[2], inflight[2], ok[2];
    for (int i = 0; i < 2; ++i) {
        inflight[i] = s->host[i].state == SLOT_INFLIGHT;
        usable[i] = s->host[i].state != SLOT_TORN_INFLIGHT;  // being torn right now: whatever it shows is going away
        if (inflight[i]) hdr[i] = s->host[i].hdr;
        else std::memcpy(&hdr[i], s->h_replica + (uint64_t)i * s->info.host_slot_stride, sizeof(hdr[i]));
    }
    const uint32_t want = full_payload(s) ? full_payload_word(s) : 0u;
    const int best = choose_slot(s, hdr, usable, want, ok);
    if (best < 0) return best;
    if (inflight[best]) PHX_CK(cudaStreamWaitEvent(st, s->ev_host[best], 0));
    rc = enqueue_restore(s, best, hdr[best], s->h_replica, s->d_replica, st, s->info.host_slot_stride, want, two_phase);
    if (rc != PHX_OK) return rc;
    for (int i = 0; i < 2; ++i) {  // adopt what the replica shows (a replacement handle starts with EMPTY slots)
        if (inflight[i] || s->host[i].state == SLOT_TORN_INFLIGHT) continue;
        s->host[i].state = ok[i] ? SLOT_COMMITTED : (s->host[i].state == SLOT_EMPTY ? SLOT_EMPTY : SLOT_TORN);
        if (ok[i]) {
            s->host[i].step = hdr[i].step;
            s->host[i].hdr = hdr[i];
        }
    }
    if (restored_step) *restored_step = s->last_step;
    return PHX_OK;
}
}  // namespace

int phx_restore(phx_shard_t *s, void *stream, uint64_t *restored_step) { return restore_own(s, stream, restored_step, false); }

// a6 in two phases: everything on `side_stream`, parameters first; see include/phx.h
int phx_restore_async(phx_shard_t *s, void *side_stream, uint64_t *restored_step)
{
    return restore_own(s, side_stream, restored_step, true);
}

int phx_restore_wait_params(phx_shard_t *s, void *stream)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    if (s->rparams_valid) PHX_CK(cudaStreamWaitEvent(static_cast<cudaStream_t>(stream), s->ev_rparams, 0));
    return PHX_OK;
}

// §8(f1): restore from a replica held elsewhere — a peer's received buffer mapped into this process
// (PAPER.md:171 stage 3, 248-250), a device buffer, or pinned host memory.  The replica is FOREIGN: this
// handle has no bookkeeping for it, so the two envelopes are read with a blocking copy (the documented
// exception to "only enqueue"; 512 bytes).
int phx_restore_from(phx_shard_t *s, const void *replica, void *stream, uint64_t *restored_step)
{
    if (!s || !replica) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    if (s->graph) return PHX_ERR_GRAPH_MODE;
    if (!aligned256(replica)) return PHX_ERR_ALIGNMENT;
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, replica);
    if (e != cudaSuccess || (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeHost) || !at.devicePointer) {
        (void)cudaGetLastError();
        return PHX_ERR_INVALID_ARG;  // pageable host memory or an unknown address
    }
    const uint8_t *r = static_cast<const uint8_t *>(replica);
    phx_snapshot_header_t hdr[2];
    const bool usable[2] = {true, true};
    bool ok[2];
    for (int i = 0; i < 2; ++i)
        PHX_CK(cudaMemcpy(&hdr[i], r + (uint64_t)i * s->info.slot_stride, sizeof(hdr[i]), cudaMemcpyDefault));
    const int best = choose_slot(s, hdr, usable, 0u, ok);
    if (best < 0) return best;
    int rc = enqueue_restore(s, best, hdr[best], r, static_cast<const uint8_t *>(at.devicePointer),
                             static_cast<cudaStream_t>(stream), s->info.slot_stride, 0u);
    if (rc == PHX_OK && restored_step) *restored_step = s->last_step;
    return rc;
}

int phx_restored_user_metadata(const phx_shard_t *s, void *blob, uint32_t cap, uint32_t *len)
{
    if (!s || (cap && !blob)) return PHX_ERR_INVALID_ARG;
    const uint32_t k = s->restored_user_len < cap ? s->restored_user_len : cap;
    if (k) std::memcpy(blob, s->restored_user, k);
    if (len) *len = s->restored_user_len;
    return PHX_OK;
}

// ---- §8(f1): peer replication around the DP ring ----------------------------------------------------
int phx_ring_peer(uint32_t dp_size, uint32_t dp_rank, int32_t j, uint32_t *peer)
{
    if (!peer || dp_size == 0 || dp_rank >= dp_size || j == 0) return PHX_ERR_INVALID_ARG;
    const int64_t a = j < 0 ? -(int64_t)j : (int64_t)j;
    if (a > (int64_t)dp_size - 1) return PHX_ERR_INVALID_ARG;  // k distinct peers need k <= D - 1
    const int64_t D = dp_size;
    *peer = (uint32_t)((((int64_t)dp_rank + j) % D + D) % D);
    return PHX_OK;
}

// Topology-aware placement (include/phx.h): the k holders of rank r's replicas are the nearest ranks
// in ring order whose failure domains differ from the owner's and from one another.
int phx_ring_peers_topology_aware(uint32_t dp_size, uint32_t dp_rank, uint32_t k, const uint32_t *domain_of_rank,
                                  uint32_t *peers)
{
    if (!domain_of_rank || (k && !peers) || dp_size == 0 || dp_rank >= dp_size || k > dp_size - 1 || k > PHX_MAX_PEERS)
        return PHX_ERR_INVALID_ARG;
    uint32_t used[PHX_MAX_PEERS + 1];
    uint32_t n_used = 0, found = 0;
    used[n_used++] = domain_of_rank[dp_rank];
    for (uint32_t j = 1; j < dp_size && found < k; ++j) {
        const uint32_t q = (dp_rank + j) % dp_size;
        bool taken = false;
        for (uint32_t u = 0; u < n_used; ++u) taken = taken || used[u] == domain_of_rank[q];
        if (taken) continue;
        used[n_used++] = domain_of_rank[q];
        peers[found++] = q;
    }
    return found == k ? PHX_OK : PHX_ERR_INVALID_ARG;  // fewer than k + 1 distinct failure domains
}

int phx_peer_buffer_alloc(uint64_t bytes, void **d_buf)
{
    if (!d_buf || bytes == 0) return PHX_ERR_INVALID_ARG;
    *d_buf = nullptr;
    void *p = nullptr;
    if (cudaMalloc(&p, bytes) != cudaSuccess) {
        (void)cudaGetLastError();
        return PHX_ERR_NOMEM;
    }
    if (cudaMemset(p, 0, bytes) != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) {
        cudaFree(p);
        return PHX_ERR_CUDA;
    }
    *d_buf = p;
    return PHX_OK;
}

int phx_peer_buffer_free(void *d_buf)
{
    if (!d_buf) return PHX_ERR_INVALID_ARG;
    return cudaFree(d_buf) == cudaSuccess ? PHX_OK : PHX_ERR_CUDA;
}

int phx_ipc_export(void *d_buf, uint8_t handle[PHX_IPC_HANDLE_BYTES])
{
    static_assert(sizeof(cudaIpcMemHandle_t) == PHX_IPC_HANDLE_BYTES, "IPC handle size");
    if (!d_buf || !handle) return PHX_ERR_INVALID_ARG;
    cudaIpcMemHandle_t h;
    if (cudaIpcGetMemHandle(&h, d_buf) != cudaSuccess) {
        (void)cudaGetLastError();
        return PHX_ERR_CUDA;
    }
    std::memcpy(handle, &h, sizeof(h));
    return PHX_OK;
}

int phx_ipc_open(const uint8_t handle[PHX_IPC_HANDLE_BYTES], void **d_buf)
{
    if (!handle || !d_buf) return PHX_ERR_INVALID_ARG;
    cudaIpcMemHandle_t h;
    std::memcpy(&h, handle, sizeof(h));
    void *p = nullptr;
    if (cudaIpcOpenMemHandle(&p, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) {
        (void)cudaGetLastError();
        return PHX_ERR_CUDA;
    }
    *d_buf = p;
    return PHX_OK;
}

int phx_ipc_close(void *d_buf)
{
    if (!d_buf) return PHX_ERR_INVALID_ARG;
    return cudaIpcCloseMemHandle(d_buf) == cudaSuccess ? PHX_OK : PHX_ERR_CUDA;
}

int phx_shard_bind_peers(phx_shard_t *s, void *const *d_peer_replicas, uint32_t k)
{
    if (!s || (k && !d_peer_replicas) || k > PHX_MAX_PEERS) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    if (!snapshots_on(s)) return PHX_ERR_SNAPSHOT_DISABLED;
    if (k > s->info.dp_size - 1) return PHX_ERR_INVALID_ARG;  // k distinct ring successors need k <= D - 1
    for (uint32_t j = 0; j < k; ++j) {
        if (!d_peer_replicas[j]) return PHX_ERR_INVALID_ARG;
        if (!aligned256(d_peer_replicas[j])) return PHX_ERR_ALIGNMENT;
        for (uint32_t i = 0; i < j; ++i)
            if (d_peer_replicas[i] == d_peer_replicas[j]) return PHX_ERR_INVALID_ARG;  // k DISTINCT peers
    }
    int rc = settle_peer_slots(s, true);
    if (rc != PHX_OK) return rc;
    if (k > 1 && !s->ev_peer_fork) PHX_CK(cudaEventCreateWithFlags(&s->ev_peer_fork, cudaEventDisableTiming));
    for (uint32_t j = 0; k > 1 && j < k; ++j) {
        if (!s->peer_st[j]) PHX_CK(cudaStreamCreateWithFlags(&s->peer_st[j], cudaStreamNonBlocking));
        if (!s->ev_peer_join[j]) PHX_CK(cudaEventCreateWithFlags(&s->ev_peer_join[j], cudaEventDisableTiming));
    }
    for (uint32_t j = 0; j < PHX_MAX_PEERS; ++j) s->d_peer[j] = j < k ? static_cast<uint8_t *>(d_peer_replicas[j]) : nullptr;
    s->n_peers = k;
    return PHX_OK;
}

int phx_snapshot_flush_peers_async(phx_shard_t *s, void *peer_stream)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound || s->n_peers == 0) return PHX_ERR_NOT_BOUND;
    if (!snapshots_on(s)) return PHX_ERR_SNAPSHOT_DISABLED;
    if (s->graph) return PHX_ERR_GRAPH_MODE;
    if (s->pending_peer_slot < 0) return PHX_ERR_NO_FLUSH_PENDING;
    cudaStream_t st = static_cast<cudaStream_t>(peer_stream);
    const int slot = s->pending_peer_slot;
    const uint64_t step = s->pending_peer_step;
    const int ps = (int)(step & 1);  // the received buffer alternates like the local pair

    PHX_CK(cudaStreamWaitEvent(st, s->ev_step[slot], 0));
    if (s->last_pflush_slot >= 0) PHX_CK(cudaStreamWaitEvent(st, s->ev_pflush[s->last_pflush_slot], 0));
    bool any_torn = false;
    for (uint32_t j = 0; j < s->n_peers; ++j) any_torn = any_torn || s->torn_peer_chunks[j] >= 0;
    s->peer[ps].step = step;
    s->peer[ps].state = any_torn ? SLOT_TORN_INFLIGHT : SLOT_INFLIGHT;
    // k = 1: the caller's stream.  k > 1: one library-owned copy stream per peer, forked from and joined back
    // into the caller's stream, so that the k transfers use k copy engines / NVLink ports at once (NVSwitch
    // gives every peer its own path; whether the source's egress then is the limit is for hardware to say).
    const bool fan = s->n_peers > 1;
    if (fan) PHX_CK(cudaEventRecord(s->ev_peer_fork, st));
    for (uint32_t j = 0; j < s->n_peers; ++j) {
        cudaStream_t pst = fan ? s->peer_st[j] : st;
        if (fan) PHX_CK(cudaStreamWaitEvent(pst, s->ev_peer_fork, 0));
        uint8_t *dst = s->d_peer[j] + (uint64_t)ps * s->info.slot_stride;
        int rc = enqueue_snapshot_copy(s, pst, dst, cudaMemcpyDefault, slot, s->torn_peer_chunks[j]);
        if (rc != PHX_OK) return rc;
        s->torn_peer_chunks[j] = -1;
        if (fan) {
            PHX_CK(cudaEventRecord(s->ev_peer_join[j], pst));
            PHX_CK(cudaStreamWaitEvent(st, s->ev_peer_join[j], 0));
        }
    }
    PHX_CK(cudaEventRecord(s->ev_pflush[slot], st));
    PHX_CK(cudaEventRecord(s->ev_peer[ps], st));
    s->pflush_valid[slot] = true;
    s->last_pflush_slot = slot;
    s->pending_peer_slot = -1;
    return PHX_OK;
}

int phx_snapshot_wait_peers(phx_shard_t *s, uint64_t step)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound || s->n_peers == 0) return PHX_ERR_NOT_BOUND;
    const int ps = (int)(step & 1);
    if (s->peer[ps].state == SLOT_EMPTY || s->peer[ps].step != step) return PHX_ERR_NO_COMMITTED_SNAPSHOT;
    int rc = settle_peer_slots(s, true);
    if (rc != PHX_OK) return rc;
    return s->peer[ps].state == SLOT_COMMITTED ? PHX_OK : PHX_ERR_CORRUPT_SLOT;
}

int phx_fault_inject_torn_peer_flush(phx_shard_t *s, uint32_t peer_j, int64_t payload_chunks)
{
    if (!s || peer_j == 0 || peer_j > PHX_MAX_PEERS) return PHX_ERR_INVALID_ARG;
    s->torn_peer_chunks[peer_j - 1] = payload_chunks < 0 ? -1 : payload_chunks;
    return PHX_OK;
}

int phx_replica_inspect(const void *replica, uint64_t slot_stride, phx_snapshot_header_t out[2], int valid[2])
{
    if (!replica || !out || !valid || slot_stride < kHeaderBytes) return PHX_ERR_INVALID_ARG;
    for (int i = 0; i < 2; ++i) {
        const uint8_t *hp = static_cast<const uint8_t *>(replica) + (uint64_t)i * slot_stride;
        if (cudaMemcpy(&out[i], hp, sizeof(out[i]), cudaMemcpyDefault) != cudaSuccess) {
            (void)cudaGetLastError();
            return PHX_ERR_CUDA;
        }
        valid[i] = header_valid(&out[i]) ? 1 : 0;
    }
    return PHX_OK;
}

// ---- §8(f3): model-parameter publication and reconstruction ---------------------------------------
int phx_shard_bind_param_peers(phx_shard_t *s, void *const *d_param_bufs, uint32_t count, uint32_t mode)
{
    if (!s || (count && !d_param_bufs) || count > PHX_MAX_PARAM_PEERS || mode > PHX_PUBLISH_COPY_ENGINE)
        return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    for (uint32_t q = 0; q < count; ++q) {
        if (!d_param_bufs[q]) return PHX_ERR_INVALID_ARG;
        if (!aligned256(d_param_bufs[q])) return PHX_ERR_ALIGNMENT;
    }
    for (uint32_t q = 0; q < PHX_MAX_PARAM_PEERS; ++q) s->d_pub[q] = q < count ? static_cast<uint8_t *>(d_param_bufs[q]) : nullptr;
    s->n_pub = count;
    s->pub_mode = mode;
    return PHX_OK;
}

int phx_publish_params_async(phx_shard_t *s, void *stream)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound || s->n_pub == 0) return PHX_ERR_NOT_BOUND;
    // ev_last_step / ev_pub are the EAGER step's events; the graph form neither records the first nor waits on the
    // second, so a publication there would wait on a stale event and race the step
    if (s->graph) return PHX_ERR_GRAPH_MODE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const uint64_t bytes = s->info.n_padded * model_elem_bytes(s);
    const uint8_t *src = fp32_mode(s) ? reinterpret_cast<const uint8_t *>(s->d_p) : static_cast<const uint8_t *>(s->d_p16);
    PHX_CK(cudaStreamWaitEvent(st, s->ev_last_step, 0));  // the newest step's kernel has written the slice
    for (uint32_t q = 0; q < s->n_pub; ++q)
        PHX_CK(cudaMemcpyAsync(s->d_pub[q] + (uint64_t)s->info.dp_rank * bytes, src, bytes, cudaMemcpyDefault, st));
    PHX_CK(cudaEventRecord(s->ev_pub, st));  // the next step (a2) and a restore wait for these reads
    s->pub_valid = true;
    return PHX_OK;
}

int phx_params_restore_from(phx_shard_t *s, const void *d_src_param_buf, void *d_dst_param_buf, void *stream)
{
    if (!s || !d_src_param_buf || !d_dst_param_buf) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    const uint64_t bytes = (uint64_t)s->info.dp_size * s->info.n_padded * model_elem_bytes(s);
    PHX_CK(cudaMemcpyAsync(d_dst_param_buf, d_src_param_buf, bytes, cudaMemcpyDefault, static_cast<cudaStream_t>(stream)));
    return PHX_OK;
}

// ---- §8(f4): full rank-state local snapshot --------------------------------------------------------
int phx_shard_bind_params(phx_shard_t *s, void *d_W)
{
    if (!s || !d_W) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    if (!aligned256(d_W)) return PHX_ERR_ALIGNMENT;
    // bf16 precision: the fused kernel keeps the rank's own range of W current through d_p_bf16
    if (!fp32_mode(s) &&
        static_cast<uint8_t *>(s->d_p16) != static_cast<uint8_t *>(d_W) + (uint64_t)s->info.dp_rank * s->info.n_padded * 2)
        return PHX_ERR_INVALID_ARG;
    s->d_W = static_cast<uint8_t *>(d_W);
    return PHX_OK;
}

int phx_params_ready(phx_shard_t *s, void *stream)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound || !s->d_W) return PHX_ERR_NOT_BOUND;
    if (s->graph) {  // graph form: the declaration is an edge of the captured graph
        const int rc = gev_record(s, s->gev_params, static_cast<cudaStream_t>(stream));
        if (rc != PHX_OK) return rc;
        s->g_params_ready = true;
        s->g_params_step = s->g_issue;
        return PHX_OK;
    }
    PHX_CK(cudaEventRecord(s->ev_params, static_cast<cudaStream_t>(stream)));
    s->params_ready = true;
    s->params_ready_step = s->last_step;
    return PHX_OK;
}

int phx_params_guard(phx_shard_t *s, void *stream)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound || !s->d_W) return PHX_ERR_NOT_BOUND;
    if (s->graph) return gev_wait(s, s->gev_wflush, static_cast<cudaStream_t>(stream));
    if (s->wflush_valid) PHX_CK(cudaStreamWaitEvent(static_cast<cudaStream_t>(stream), s->ev_wflush, 0));
    return PHX_OK;
}

// ---- introspection -----------------------------------------------------------------------------
int phx_last_step(const phx_shard_t *s, uint64_t *step)
{
    if (!s || !step) return PHX_ERR_INVALID_ARG;
    *step = s->last_step;
    return PHX_OK;
}

// ---- §8(e): global clip, a1 split around the caller's exchange ------------------------------------
int phx_grad_sumsq_async(phx_shard_t *s, const void *d_grads, double *d_out, void *stream)
{
    if (!s || !d_grads || !d_out) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    if (!aligned256(d_grads) || (reinterpret_cast<uintptr_t>(d_out) & 7u)) return PHX_ERR_ALIGNMENT;
    int nl = 0;
    PHX_CK(phx::launch_sumsq(d_grads, fp32_mode(s), s->info.n_padded, s->d_partials, d_out,
                             static_cast<cudaStream_t>(stream), &nl));
    s->launches += nl;
    return PHX_OK;
}

int phx_set_clip_partials(phx_shard_t *s, const double *d_partials, uint32_t count)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (d_partials == nullptr) {
        s->clip_partials = nullptr;
        s->clip_count = 0;
        return PHX_OK;
    }
    if (!(s->cfg.max_grad_norm > 0.0f) || count < 1 || count > (uint32_t)phx::kSumsqMaxBlocks) return PHX_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(d_partials) & 7u) return PHX_ERR_ALIGNMENT;
    s->clip_partials = d_partials;
    s->clip_count = count;
    return PHX_OK;
}

int phx_last_clip(phx_shard_t *s, float *coef, double *sumsq)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    if (s->graph) return PHX_ERR_GRAPH_MODE;  // it would synchronise on the last EAGER step's event, not on the replay
    float c = 1.0f;
    double q = 0.0;
    if (s->clip_valid) {
        PHX_CK(cudaEventSynchronize(s->ev_last_step));  // the step that used it has run
        PHX_CK(cudaMemcpy(&c, s->d_scratch + kScrCoef, 4, cudaMemcpyDeviceToHost));
        PHX_CK(cudaMemcpy(&q, s->d_scratch + kScrSumsq, 8, cudaMemcpyDeviceToHost));
    }
    if (coef) *coef = c;
    if (sumsq) *sumsq = q;
    return PHX_OK;
}

int phx_kernel_launches(const phx_shard_t *s, uint64_t *count)
{
    if (!s || !count) return PHX_ERR_INVALID_ARG;
    *count = s->launches;
    return PHX_OK;
}

int phx_dropped_snapshots(const phx_shard_t *s, uint64_t *host, uint64_t *peers)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (host) *host = s->dropped_host;
    if (peers) *peers = s->dropped_peers;
    return PHX_OK;
}

// ---- §8(f4), second half: the gradient producer's epilogue ------------------------------------------
int phx_grads_finalize_async(phx_shard_t *s, const float *d_main_grads_fp32, float scale, void *d_grads_bf16_out,
                             double *d_sumsq_out, void *stream)
{
    if (!s || !d_main_grads_fp32 || !d_grads_bf16_out || !d_sumsq_out || !(scale == scale)) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    if (fp32_mode(s)) return PHX_ERR_INVALID_ARG;  // the all-FP32 precision has no bf16 gradients to produce
    if (!aligned256(d_main_grads_fp32) || !aligned256(d_grads_bf16_out) || (reinterpret_cast<uintptr_t>(d_sumsq_out) & 7u))
        return PHX_ERR_ALIGNMENT;
    const uint64_t N = s->info.n_padded;
    const uint8_t *in0 = reinterpret_cast<const uint8_t *>(d_main_grads_fp32), *out0 = static_cast<const uint8_t *>(d_grads_bf16_out);
    if (in0 < out0 + 2 * N && out0 < in0 + 4 * N) return PHX_ERR_INVALID_ARG;  // the two arrays must not overlap
    int nl = 0;
    PHX_CK(phx::launch_grads_finalize(d_main_grads_fp32, scale, d_grads_bf16_out, N,
                                      s->d_partials + phx::sumsq_partials_count(N), d_sumsq_out,
                                      static_cast<cudaStream_t>(stream), &nl));
    s->launches += nl;
    return PHX_OK;
}

// ---- derived scalars, exposed for the tests that pin them to the oracle ------------------------------
int phx_derived_scalars_host(float lr, float beta1, float beta2, float wd, uint64_t step, float out[5])
{
    if (!out || step == 0) return PHX_ERR_INVALID_ARG;
    phx::AdamScalars sc;
    derive_scalars_host(lr, beta1, beta2, 0.0f, wd, step, &sc);
    out[0] = sc.decay, out[1] = sc.omb1, out[2] = sc.omb2, out[3] = sc.ss, out[4] = sc.sbc2;
    return PHX_OK;
}

int phx_derived_scalars_device(float lr, float beta1, float beta2, float wd, const uint64_t *steps, uint32_t n, float *out)
{
    if ((!steps || !out) && n) return PHX_ERR_INVALID_ARG;
    if (n == 0) return PHX_OK;
    uint64_t *d_steps = nullptr;
    float *d_out = nullptr;
    int rc = PHX_OK;
    if (cudaMalloc(reinterpret_cast<void **>(&d_steps), (size_t)n * 8) != cudaSuccess ||
        cudaMalloc(reinterpret_cast<void **>(&d_out), (size_t)n * 20) != cudaSuccess)
        rc = PHX_ERR_NOMEM;
    if (rc == PHX_OK &&
        (cudaMemcpy(d_steps, steps, (size_t)n * 8, cudaMemcpyHostToDevice) != cudaSuccess ||
         phx::launch_derive_scalars(lr, beta1, beta2, wd, d_steps, n, d_out, nullptr) != cudaSuccess ||
         cudaMemcpy(out, d_out, (size_t)n * 20, cudaMemcpyDeviceToHost) != cudaSuccess))
        rc = PHX_ERR_CUDA;
    if (rc != PHX_OK) (void)cudaGetLastError();
    cudaFree(d_steps);
    cudaFree(d_out);
    return rc;
}

// ---- the graph-capturable form (include/phx.h "graph") -----------------------------------------------
namespace {
phx::StepBlock *step_block(phx_shard *s) { return reinterpret_cast<phx::StepBlock *>(s->d_scratch + kScrBlock); }
}  // namespace

int phx_graph_begin(phx_shard_t *s, float lr, float beta1, float beta2, float eps, float wd, void *stream)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    if (s->graph) return PHX_ERR_GRAPH_MODE;
    if (full_payload(s) && !s->d_W) return PHX_ERR_NOT_BOUND;
    // a mode switch, not a hot call: every eager flush of this handle lands before the first captured / replayed
    // step may touch what it reads
    int rc = settle_host_slots(s, true);
    if (rc != PHX_OK) return rc;
    rc = settle_peer_slots(s, true);
    if (rc != PHX_OK) return rc;
    if (s->rstate_valid) {  // a two-phase restore still bringing the moments back
        PHX_CK(cudaEventSynchronize(s->ev_rstate));
        s->rstate_valid = false;
    }
    phx_snapshot_header_t tmpl;
    build_header(s, 0, true, &tmpl);
    phx::HeaderBlob blob;
    std::memcpy(&blob, &tmpl, sizeof(blob));
    PHX_CK(phx::launch_step_block_init(step_block(s), lr, beta1, beta2, eps, wd, s->last_step, blob,
                                       static_cast<cudaStream_t>(stream)));
    s->launches += 1;
    s->graph = true;
    s->g_issue = s->last_step;
    s->g_pending_slot = s->pending_slot;   // an eager step's un-flushed snapshot becomes the graph's first flush
    s->g_pending_step = s->pending_step;
    s->g_last_flush_slot = -1;
    s->g_pending_peer_slot = s->n_peers ? s->pending_peer_slot : -1;
    s->g_pending_peer_step = s->pending_peer_step;
    s->g_last_pflush_slot = -1;
    for (int k = 0; k < kMaxDepth; ++k) s->gev_step[k].valid = s->gev_flush[k].valid = s->gev_pflush[k].valid = false;
    s->gev_params.valid = s->gev_wflush.valid = false;
    // an eager declaration for the pending snapshot carries over (the eager events have all been settled above)
    s->g_params_ready = s->params_ready;
    s->g_params_step = s->params_ready_step;
    return PHX_OK;
}

int phx_graph_set_hyper(phx_shard_t *s, float lr, float beta1, float beta2, float eps, float wd, void *stream)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    if (!s->graph) return PHX_ERR_GRAPH_MODE;
    // Not capturable: the source is a host stack array.  Outside a capture cudaMemcpyAsync stages a pageable source
    // before it returns; a captured memcpy node would keep the dangling pointer and read it at every replay.
    if (capture_id(static_cast<cudaStream_t>(stream)) != 0) return PHX_ERR_INVALID_ARG;
    // five floats at the front of the block's hyperparameter area, stream-ordered; the step counter stays
    const float h[5] = {lr, beta1, beta2, eps, wd};
    PHX_CK(cudaMemcpyAsync(reinterpret_cast<uint8_t *>(step_block(s)) + offsetof(phx::StepBlock, lr), h, sizeof(h),
                           cudaMemcpyHostToDevice, static_cast<cudaStream_t>(stream)));
    return PHX_OK;
}

// The caller blob of the envelope (RNG states) changes every iteration; in the graph form the envelope
// template lives in the device step block, so the update is a stream-ordered copy into it (user_len ‖ payload ‖
// user[128] are contiguous in phx_snapshot_header_t; the prologue rewrites the payload word per slot anyway).
int phx_graph_set_user_metadata(phx_shard_t *s, const void *blob, uint32_t len, void *stream)
{
    if (!s || len > 128 || (len && !blob)) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    if (!s->graph) return PHX_ERR_GRAPH_MODE;
    if (capture_id(static_cast<cudaStream_t>(stream)) != 0) return PHX_ERR_INVALID_ARG;  // pageable source, see set_hyper
    std::memset(s->user, 0, sizeof(s->user));
    if (len) std::memcpy(s->user, blob, len);
    s->user_len = len;  // the eager calls after phx_graph_end carry the same blob on
    phx_snapshot_header_t tmpl;
    build_header(s, 0, true, &tmpl);
    constexpr size_t off = offsetof(phx_snapshot_header_t, user_len);
    constexpr size_t bytes = offsetof(phx_snapshot_header_t, user) + sizeof(tmpl.user) - off;
    static_assert(bytes == 136, "user_len, payload and user[] are contiguous");
    PHX_CK(cudaMemcpyAsync(reinterpret_cast<uint8_t *>(step_block(s)) + offsetof(phx::StepBlock, hdr_tmpl) + off,
                           reinterpret_cast<const uint8_t *>(&tmpl) + off, bytes, cudaMemcpyHostToDevice,
                           static_cast<cudaStream_t>(stream)));
    return PHX_OK;
}

int phx_graph_step_and_snapshot(phx_shard_t *s, const void *d_grads, void *stream)
{
    if (!s || !d_grads) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    if (!s->graph) return PHX_ERR_GRAPH_MODE;
    if (int rcd = check_device(s)) return rcd;
    if (!aligned256(d_grads)) return PHX_ERR_ALIGNMENT;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const bool snap = snapshots_on(s);
    const uint64_t step = s->g_issue + 1;  // issue order; on a replay the device counter is the truth

    phx::StepArgs a;
    std::memset(&a, 0, sizeof(a));
    int rc = enqueue_clip(s, d_grads, a, st);
    if (rc != PHX_OK) return rc;
    int slot = -1;
    const uint32_t depth = ring_depth(s);
    if (snap) {
        slot = (int)(step % depth);
        // a2, the single sync point: a dependency edge inside a captured graph, a stream wait outside
        if (s->cfg.sync_mode == PHX_SYNC_STRICT) {
            if (s->g_last_flush_slot >= 0 && (rc = gev_wait(s, s->gev_flush[s->g_last_flush_slot], st)) != PHX_OK) return rc;
            if (s->g_last_pflush_slot >= 0 && (rc = gev_wait(s, s->gev_pflush[s->g_last_pflush_slot], st)) != PHX_OK) return rc;
        } else {
            if ((rc = gev_wait(s, s->gev_flush[slot], st)) != PHX_OK) return rc;
            if ((rc = gev_wait(s, s->gev_pflush[slot], st)) != PHX_OK) return rc;
            // §8(f4): the kernel rewrites this rank's range of W, which the newest full-rank-state flush reads
            if (full_payload(s) && (rc = gev_wait(s, s->gev_wflush, st)) != PHX_OK) return rc;
        }
        if (s->g_pending_slot >= 0 && s->h_replica) s->dropped_host += 1;
        if (s->g_pending_peer_slot >= 0 && s->n_peers) s->dropped_peers += 1;
    }
    fill_common_args(s, d_grads, slot, a);
    void *shdr = a.shdr;
    a.shdr = nullptr;  // the prologue writes the envelope; the fused kernel only moves elements
    a.dsc = &step_block(s)->sc;
    void *shdr_full = nullptr;
    uint32_t full_word = 0u;
    if (snap && full_payload(s)) {  // §8(f4): the local slot's envelope differs in the payload word and the hash
        shdr_full = s->d_scratch + kScrHdrFull + (size_t)slot * kHeaderBytes;
        full_word = full_payload_word(s);
    }
    // What a captured call bakes in: the staging slot (step mod depth) AND the host / peer ping-pong slot (step mod 2,
    // phx_graph_flush_async).  The device check therefore runs modulo lcm(depth, 2): with depth 1 or 3 a replay can land
    // on the right staging slot and still on the wrong host slot (it would invalidate and rewrite the newest committed
    // replica), which the staging-slot test alone let through.
    const uint32_t period = (depth & 1u) ? 2u * depth : depth;
    PHX_CK(phx::launch_step_prologue(step_block(s), shdr, shdr_full, full_word, snap ? (uint32_t)(step % period) : 0u,
                                     snap ? period : 0u, st));
    PHX_CK(phx::launch_step(a, snap && !direct_mode(s), step_mode(s), true, st));
    s->launches += 1 + (s->info.n_padded ? 1 : 0);
    if (snap) {
        if ((rc = gev_record(s, s->gev_step[slot], st)) != PHX_OK) return rc;
        s->g_pending_slot = slot;
        s->g_pending_step = step;
        if (s->n_peers) {
            s->g_pending_peer_slot = slot;
            s->g_pending_peer_step = step;
        }
    }
    s->g_issue = step;
    s->g_params_ready = false;
    return PHX_OK;
}

int phx_graph_flush_async(phx_shard_t *s, void *side_stream)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound || (snapshots_on(s) && !s->h_replica)) return PHX_ERR_NOT_BOUND;
    if (!snapshots_on(s)) return PHX_ERR_SNAPSHOT_DISABLED;
    if (!s->graph) return PHX_ERR_GRAPH_MODE;
    if (int rcd = check_device(s)) return rcd;
    if (s->g_pending_slot < 0) return PHX_ERR_NO_FLUSH_PENDING;
    cudaStream_t st = static_cast<cudaStream_t>(side_stream);
    const int slot = s->g_pending_slot;
    const int hs = (int)(s->g_pending_step & 1);  // ping-pong; kept on a replay by the alignment rule
    uint8_t *dst = s->h_replica + (uint64_t)hs * s->info.host_slot_stride;
    int rc;
    const bool full = full_payload(s);
    if (full) {
        if (!s->d_W) return PHX_ERR_NOT_BOUND;
        if (!s->g_params_ready || s->g_params_step != s->g_pending_step) return PHX_ERR_PARAMS_NOT_READY;
        if ((rc = gev_wait(s, s->gev_params, st)) != PHX_OK) return rc;  // the all-gather of this step has landed in W
    }
    if ((rc = gev_wait(s, s->gev_step[slot], st)) != PHX_OK) return rc;  // the step's kernel has written the slot
    if (s->g_last_flush_slot >= 0 && (rc = gev_wait(s, s->gev_flush[s->g_last_flush_slot], st)) != PHX_OK) return rc;
    rc = enqueue_snapshot_copy(s, st, dst, cudaMemcpyDeviceToHost, slot, -1, full, full ? &s->gev_wflush : nullptr);
    if (rc != PHX_OK) return rc;
    if ((rc = gev_record(s, s->gev_flush[slot], st)) != PHX_OK) return rc;
    s->g_last_flush_slot = slot;
    s->g_pending_slot = -1;
    return PHX_OK;
}

// §8(f1) in the graph form: the replication of the last issued step's snapshot to the k ring peers, capturable
int phx_graph_flush_peers_async(phx_shard_t *s, void *peer_stream)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound || s->n_peers == 0) return PHX_ERR_NOT_BOUND;
    if (!snapshots_on(s)) return PHX_ERR_SNAPSHOT_DISABLED;
    if (!s->graph) return PHX_ERR_GRAPH_MODE;
    if (s->g_pending_peer_slot < 0) return PHX_ERR_NO_FLUSH_PENDING;
    cudaStream_t st = static_cast<cudaStream_t>(peer_stream);
    const int slot = s->g_pending_peer_slot;
    const int ps = (int)(s->g_pending_peer_step & 1);
    int rc;
    if ((rc = gev_wait(s, s->gev_step[slot], st)) != PHX_OK) return rc;
    if (s->g_last_pflush_slot >= 0 && (rc = gev_wait(s, s->gev_pflush[s->g_last_pflush_slot], st)) != PHX_OK) return rc;
    const bool fan = s->n_peers > 1;  // one library-owned copy stream per peer, forked from and joined into `st`
    if (fan) PHX_CK(cudaEventRecord(s->ev_peer_fork, st));
    for (uint32_t j = 0; j < s->n_peers; ++j) {
        cudaStream_t pst = fan ? s->peer_st[j] : st;
        if (fan) PHX_CK(cudaStreamWaitEvent(pst, s->ev_peer_fork, 0));
        rc = enqueue_snapshot_copy(s, pst, s->d_peer[j] + (uint64_t)ps * s->info.slot_stride, cudaMemcpyDefault, slot, -1);
        if (rc != PHX_OK) return rc;
        if (fan) {
            PHX_CK(cudaEventRecord(s->ev_peer_join[j], pst));
            PHX_CK(cudaStreamWaitEvent(st, s->ev_peer_join[j], 0));
        }
    }
    if ((rc = gev_record(s, s->gev_pflush[slot], st)) != PHX_OK) return rc;
    s->g_last_pflush_slot = slot;
    s->g_pending_peer_slot = -1;
    return PHX_OK;
}

int phx_graph_end(phx_shard_t *s, uint64_t *last_step)
{
    if (!s) return PHX_ERR_INVALID_ARG;
    if (!s->bound) return PHX_ERR_NOT_BOUND;
    if (!s->graph) return PHX_ERR_GRAPH_MODE;
    PHX_CK(cudaDeviceSynchronize());  // mode switch: every replay and every flush has finished
    phx::StepBlock blk;
    PHX_CK(cudaMemcpy(&blk, step_block(s), sizeof(blk), cudaMemcpyDeviceToHost));
    s->graph = false;
    s->last_step = blk.step;
    // the eager bookkeeping restarts from what is self-describing: the envelopes in the host slots
    for (int k = 0; k < kMaxDepth; ++k) s->flush_valid[k] = s->pflush_valid[k] = false;
    s->wflush_valid = false;  // nothing is reading W any more (device synchronised above)
    // g_params_step counts ISSUED calls (the host mirror), blk.step is the device counter, which runs ahead of it
    // after any replay: a declaration made for the last issued step holds for the step the device finished last
    // (in a replayed graph the declaration is an edge behind that step's kernel), so it carries over.
    s->params_ready = s->g_params_ready && s->g_params_step == s->g_issue;
    s->params_ready_step = s->params_ready ? blk.step : 0;
    s->last_flush_slot = s->last_pflush_slot = -1;
    s->pending_slot = s->pending_peer_slot = -1;
    uint64_t newest = 0;
    for (int i = 0; i < 2 && s->h_replica; ++i) {
        phx_snapshot_header_t h;
        std::memcpy(&h, s->h_replica + (uint64_t)i * s->info.host_slot_stride, sizeof(h));
        const bool ok = header_valid(&h) && header_matches(s, &h) && h.payload == (full_payload(s) ? full_payload_word(s) : 0u);
        s->host[i].state = ok ? SLOT_COMMITTED : SLOT_EMPTY;
        s->host[i].step = ok ? h.step : 0;
        if (ok) s->host[i].hdr = h;
        if (ok && h.step > newest) newest = h.step;
    }
    if (snapshots_on(s) && s->last_step > 0 && newest != s->last_step) {  // the newest step's snapshot is still staged
        s->pending_slot = (int)(s->last_step % ring_depth(s));
        s->pending_step = s->last_step;
    }
    // the peers' slots are self-describing too: the first peer's two envelopes (all k peers are written as one unit)
    uint64_t newest_peer = 0;
    for (int i = 0; i < 2; ++i) {
        s->peer[i].state = SLOT_EMPTY;
        if (!s->n_peers) continue;
        phx_snapshot_header_t h;
        PHX_CK(cudaMemcpy(&h, s->d_peer[0] + (uint64_t)i * s->info.slot_stride, sizeof(h), cudaMemcpyDefault));
        if (!(header_valid(&h) && header_matches(s, &h) && h.payload == 0u)) continue;
        s->peer[i].state = SLOT_COMMITTED;
        s->peer[i].step = h.step;
        if (h.step > newest_peer) newest_peer = h.step;
    }
    if (snapshots_on(s) && s->n_peers && s->last_step > 0 && newest_peer != s->last_step) {
        s->pending_peer_slot = (int)(s->last_step % ring_depth(s));
        s->pending_peer_step = s->last_step;
    }
    if (last_step) *last_step = s->last_step;
    return blk.misaligned ? PHX_ERR_STEP_ORDER : PHX_OK;
}

}  // extern "C"
