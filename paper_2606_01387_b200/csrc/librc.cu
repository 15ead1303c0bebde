// librc.cu -- host side of librc: the C ABI of include/rc.h, the claim table, the extent
// allocators (block-table arena, digest arena, pinned host store) and the transfer engine
// (staging rings, gather/scatter streams, copy streams, events).  Every step of the path runs in
// the kernels of rc_kernels.cuh or on the copy engines; the host only validates arguments,
// orders the work and mirrors claim state.  There is no CPU fallback: without a CUDA device
// rc_create fails with RC_ERR_CUDA.
//
// Ordering model: metadata kernels (accept, predicate, plan/allocation,
// reference drops, verdicts, event emission) all run on ONE in-order stream, `meta`, in call
// order; bulk movement runs on (gather, d2h) for offload and (scatter, h2d) for restore and is
// fenced to `meta` with events.  So an offload and a restore may overlap their data movement
// while every observable result equals the synchronous calls in _begin order.
#include "../../include/rc.h"
#include "rc_kernels.cuh"
#include "rc_trace.cuh"

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <unordered_map>
#include <unordered_set>
#include <vector>

using namespace rck;

namespace {

// first-fit extent allocator over [0, cap) units; free extents kept merged in address order
struct ExtAlloc {
  std::map<u64, u64> fr;
  u64 cap = 0, free_total = 0;
  void init(u64 c) { fr.clear(); cap = free_total = c; if (c) fr[0] = c; }
  bool alloc(u64 n, u64& off) {
    if (n == 0) { off = 0; return true; }
    for (auto it = fr.begin(); it != fr.end(); ++it)
      if (it->second >= n) {
        off = it->first;
        const u64 rest = it->second - n;
        fr.erase(it);
        if (rest) fr[off + n] = rest;
        free_total -= n;
        return true;
      }
    return false;
  }
  // n units in as few pieces as the free list allows, lowest addresses first (never fails when
  // free_total >= n: the host store is granted by byte count, not by contiguity)
  bool alloc_split(u64 n, std::vector<std::pair<u64, u64>>& out) {
    if (n > free_total) return false;
    u64 o;
    if (alloc(n, o)) { out.push_back({o, n}); return true; }
    while (n) {
      auto it = fr.begin();
      const u64 take = std::min(n, it->second), at = it->first, rest = it->second - take;
      fr.erase(it);
      if (rest) fr[at + take] = rest;
      free_total -= take;
      out.push_back({at, take});
      n -= take;
    }
    return true;
  }
  void release(u64 off, u64 n) {
    if (!n) return;
    auto nx = fr.lower_bound(off);
    if (nx != fr.begin()) {
      auto pv = std::prev(nx);
      if (pv->first + pv->second == off) { off = pv->first; n += pv->second; fr.erase(pv); }
    }
    if (nx != fr.end() && off + n == nx->first) { n += nx->second; fr.erase(nx); }
    fr[off] = n;
    free_total += (n - 0);
  }
};

typedef std::pair<u64, u64> Key;          // 128-bit content key of a block: (checksum d, second digest e)
struct KeyHash { size_t operator()(const Key& k) const { return (size_t)(k.first ^ (k.second * 0x9E3779B97F4A7C15ull)); } };

struct Claim {
  u64 id = 0, chain = 0;
  u32 state = 0, P = 0, N = 0, M = 0, nb = 0, policy = 0;
  u32 protect = 0;                       // NEXT-3: hard_protected -- never a victim of rc_make_room
  u64 order = 0;                         // acceptance sequence number: the victim order
  u32 bt_off = 0, bt_len = 0;            // live table extent (bt_len == 0: no table)
  u32 dg_off = 0, dg_len = 0;            // recorded digests
  std::vector<std::pair<u64, u64>> host; // host-store extents in blk units
  std::vector<u32> hslots;               // dedup mode: host-store slot of each block
  std::vector<Key> hkeys;                // dedup mode: 128-bit content key (d, e) of each block
  bool busy = false;
};

struct Seg { u64 w0, n, hoff; };          // n blocks at work position w0 <-> host-store block hoff

struct Op {
  bool active = false;
  u32 n = 0;
  int32_t* status = nullptr;
  std::vector<Claim*> cl;                 // per batch entry: served claim or nullptr
  std::vector<u32> new_bt;                // restore: new table extent offset per entry
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> t_kernel, t_copy;
  u64 blocks = 0, copy_bytes = 0, launches = 0;
  // restore: the reuse request it belongs to (0: per-claim refusals), TP split form, verdict kernels already enqueued
  u64 request_id = 0; bool tp = false, tail = false;
};

}  // namespace

struct rc_ctx {
  rc_config cfg;
  u32 G = 0, vpp = 0, NB = 0, R = 0, sms = 0, grid = 0, mover = 0;
  u32 tma_variant[3] = {0, 0, 0}, tma_grid[3] = {0, 0, 0};   // per mover mode (gather, scatter, digest)
  u64 page = 0, blk = 0, chunk_blocks = 0, host_blocks = 0, cap_entries = 0, desc_cap = 0;
  cudaStream_t meta = 0, gather = 0, d2h = 0, scatter = 0, h2d = 0, util = 0;
  bool own[5] = {false, false, false, false, false};
  u8* pool = nullptr; u8* fill = nullptr;
  u8* d_used = nullptr; u32* d_ref = nullptr; u32* d_bt = nullptr; u64* d_dg = nullptr; u64* d_dg2 = nullptr;
  Event* h_evbuf = nullptr; u64 ev_bounce_cap = 0;         // rc_outcomes: mapped pinned bounce buffer
  Event* d_ring = nullptr; u64* d_evcount = nullptr; u32* d_bitmaps = nullptr; u32* d_up = nullptr;
  u32* d_counters = nullptr; u32* d_alloc = nullptr; u64* d_flip = nullptr;
  u32 *d_posmax = nullptr, *d_gain = nullptr; u8* d_protmap = nullptr; u64 accept_seq = 0;   // NEXT-3 allocator-side protection
  // NEXT-4: TP-sharded KV.  Mailbox = [TP_MAX_RANKS epoch flags][G x desc_cap verdict records], peer-writable.
  u32 tp_ranks = 0, tp_rank = 0, tp_n = 0; bool tp_split = false, tp_pending = false; u64 tp_epoch = 0;
  u8* d_mailbox = nullptr; u64 mailbox_bytes = 0; TpVerdict *d_verd = nullptr, *d_gath = nullptr, *h_verd = nullptr;
  u8* peer_mb[TP_MAX_RANKS] = {}; bool peer_ipc[TP_MAX_RANKS] = {};
  // descriptor / result sets: 0 = offload slot 0, 1 = restore, 2 = the synchronous metadata calls, 3 = offload slot 1
  Desc* d_desc[4] = {}; Res* d_res[4] = {}; u32* d_off[4] = {};
  Desc* h_desc[4] = {}; Res* h_res[4] = {};
  u32* h_up = nullptr; u64* h_flip = nullptr; u32* h_counters = nullptr;
  bool check = false; u32 *h_check = nullptr, *d_check = nullptr;   // RC_CHECK=1: work items validated before every mover launch
  // per operation in flight: work list and block digests.  Index = op index: 0 = offload slot 0, 1 = restore, 2 = offload slot 1
  u32* d_phys[3] = {}; u64* d_dtmp[3] = {}; u64* d_etmp[3] = {};
  std::vector<u8*> staging[2]; std::vector<u64*> part[2];
  std::vector<cudaEvent_t> ev_free[2], ev_ready[2];
  std::vector<bool> slot_used[2];
  cudaEvent_t ev_plan[2] = {}, ev_body_a[3] = {}, ev_body_b[3] = {};   // ev_body_*: by op index
  u64 chunk_seq[2] = {0, 0};                               // staging ring position per direction, running across operations
  std::vector<cudaEvent_t> ev_pool;
  u8* h_store = nullptr;
  ExtAlloc host_alloc, bt_alloc, dg_alloc;
  u64 host_used = 0;
  std::unordered_map<u64, Claim> claims;
  std::vector<rc_fault> faults; u32 fault_flags = 0;
  u64 ev_emitted = 0, ev_drained = 0, ev_reserved = 0;
  rc_stats st;
  Op ops[3];                                               // by op index (above)
  int off_q[2] = {0, 0}; int off_open = 0;                 // offloads begun and not yet completed by rc_wait(0), oldest first
  bool poisoned = false;
  std::string cuda_err;
  int accept_ctas = 32;
  // NEXT-2: content-addressed host store
  u64 request_id = 0;                                    // NEXT-3: the reuse request of the restore being begun (0: per-claim)
  bool dedup = false;
  std::unordered_map<Key, std::pair<u32, u32>, KeyHash> store;   // (d, e) -> (slot, references)
  u64 *h_dig = nullptr, *h_dig2 = nullptr; u32 *h_iw = nullptr, *h_ispos = nullptr, *d_iw = nullptr, *d_ispos = nullptr;
  // NEXT-4 (first half): gather straight into the mapped pinned store, no staging, no copy engine
  bool lm = false;                                       // NEXT-4: layer-major host copy and chunk layout (rc.h)
  bool direct = false; u8* h_store_dev = nullptr; u32 *h_hpos = nullptr, *d_hpos = nullptr;
};

#define CK(call)                                                                      \
  do {                                                                                \
    cudaError_t e_ = (call);                                                          \
    if (e_ != cudaSuccess) {                                                          \
      c->poisoned = true;                                                             \
      c->cuda_err = std::string(#call) + ": " + cudaGetErrorString(e_);               \
      return RC_ERR_CUDA;                                                             \
    }                                                                                 \
  } while (0)
#define CKL() CK(cudaGetLastError())

static inline u32 ceil_div(u32 a, u32 b) { return (a + b - 1) / b; }
static inline u32 warps_grid(u32 n) { return (n * 32 + 255) / 256; }

static cudaEvent_t get_event(rc_ctx* c) {
  if (!c->ev_pool.empty()) { cudaEvent_t e = c->ev_pool.back(); c->ev_pool.pop_back(); return e; }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}

// ---- small transfers ----------------------------------------------------------------------------------------
// host_ptr is a mapped pinned buffer of the library (cudaHostAllocMapped); the words cross PCIe in a kernel on `s`, in
// stream order, never through a copy engine (rc_kernels.cuh: k_copy_words).  bytes % 4 == 0.
static cudaError_t small_copy(rc_ctx* c, cudaStream_t s, void* dst, const void* src, u64 bytes, bool dst_is_host) {
  if (!bytes) return cudaSuccess;
  void* hd = nullptr;
  cudaError_t e = cudaHostGetDevicePointer(&hd, dst_is_host ? dst : const_cast<void*>(src), 0);
  if (e != cudaSuccess) return e;
  const u64 n = bytes / 4;
  const u32 grid = (u32)std::min<u64>((n + 255) / 256, 592);
  if (dst_is_host) k_copy_words<<<grid, 256, 0, s>>>((u32*)hd, (const u32*)src, n);
  else k_copy_words<<<grid, 256, 0, s>>>((u32*)dst, (const u32*)hd, n);
  c->st.kernel_launches++;
  return cudaGetLastError();
}
static inline cudaError_t to_dev(rc_ctx* c, cudaStream_t s, void* d, const void* h, u64 bytes) { return small_copy(c, s, d, h, bytes, false); }
static inline cudaError_t to_host(rc_ctx* c, cudaStream_t s, void* h, const void* d, u64 bytes) { return small_copy(c, s, h, d, bytes, true); }

// ---- data movers -----------------------------------------------------------------------------
template <int MODE>
static void launch_ldg(rc_ctx* c, cudaStream_t s, u8* staging, const u32* phys, u64* part, u32 n_items, const u32* iw, const u32* ispos,
                       u32 sw, u32 sg) {
  const u32 pages = n_items * c->G;
  const u32 grid = std::min(pages, c->grid);
  const u32 vpt = c->vpp / LANES;
  if (vpt % 8 == 0)
    k_move_hash<MODE, 8><<<grid, LANES, 0, s>>>((uint4*)c->pool, (uint4*)staging, phys, part, n_items, c->G, c->NB, c->vpp, iw, ispos, sw, sg);
  else if (vpt % 4 == 0)
    k_move_hash<MODE, 4><<<grid, LANES, 0, s>>>((uint4*)c->pool, (uint4*)staging, phys, part, n_items, c->G, c->NB, c->vpp, iw, ispos, sw, sg);
  else
    k_move_hash<MODE, 1><<<grid, LANES, 0, s>>>((uint4*)c->pool, (uint4*)staging, phys, part, n_items, c->G, c->NB, c->vpp, iw, ispos, sw, sg);
}

// (TILE, STAGES per group, consumer groups, CTAs/SM) variants of the TMA mover; RC_TMA_VARIANT=<index> overrides the
// default choice (tuning sweeps, profiles/r02_mover_sweep.md)
typedef void (*tma_fn)(u8*, u8*, const u32*, u64*, u32, u32, u32, u32, const u32*, const u32*, u32, u32);
struct TmaVariant { u32 tile, stages, groups, ctas_per_sm; tma_fn fn[3]; };
#define TMA_V(T, S, NG, C) {T, S, NG, C, {k_move_hash_tma<MV_GATHER, S, T, NG>, k_move_hash_tma<MV_SCATTER, S, T, NG>, k_move_hash_tma<MV_DIGEST, S, T, NG>}}
static const TmaVariant kTma[] = {
    TMA_V(4096, 4, 1, 2),  TMA_V(8192, 4, 1, 2),  TMA_V(8192, 8, 1, 1),   TMA_V(16384, 3, 1, 2),  TMA_V(16384, 4, 1, 1),
    TMA_V(16384, 6, 1, 1), TMA_V(32768, 2, 1, 2), TMA_V(32768, 3, 1, 1),  TMA_V(16384, 12, 1, 1), TMA_V(32768, 6, 1, 1),
    /* 10.. two consumer groups */
    TMA_V(32768, 2, 2, 1), TMA_V(32768, 3, 2, 1), TMA_V(16384, 3, 2, 1),  TMA_V(16384, 4, 2, 1),  TMA_V(16384, 6, 2, 1),
    TMA_V(16384, 2, 2, 2), TMA_V(16384, 3, 2, 2), TMA_V(8192, 4, 2, 2),   TMA_V(4096, 4, 2, 2),   TMA_V(32768, 4, 1, 1),
    /* 20.. small tiles */
    TMA_V(8192, 3, 1, 2),  TMA_V(8192, 6, 1, 1),  TMA_V(8192, 4, 1, 3),   TMA_V(16384, 2, 1, 2),  TMA_V(4096, 8, 1, 2),
    TMA_V(8192, 2, 1, 4),  TMA_V(8192, 6, 1, 2),  TMA_V(4096, 6, 1, 3),   TMA_V(8192, 3, 2, 2),   TMA_V(8192, 2, 2, 2)};
constexpr int kTmaN = sizeof(kTma) / sizeof(kTma[0]);
static inline u32 tma_smem(const TmaVariant& v) { return v.tile * v.stages * v.groups; }
static inline u32 tma_block(const TmaVariant& v) { return v.groups * LANES + 64; }

template <int MODE>
static void launch_move(rc_ctx* c, cudaStream_t s, u8* staging, const u32* phys, u64* part, u32 n_items,
                        const u32* iw = nullptr, const u32* ispos = nullptr, bool layer_major = false) {
  const u32 sw = layer_major ? 1u : c->G, sg = layer_major ? n_items : 1u;     // staged page of (item, g): w*sw + g*sg
  if (c->check) {                                          // RC_CHECK=1: bound every access of this launch by its work items
    const bool to_host_store = c->direct && staging == c->h_store_dev;
    const u64 staged_limit = to_host_store ? c->host_blocks : c->chunk_blocks;
    if (n_items > c->chunk_blocks) *c->h_check = 1u;      // the partial-sum buffer and a staging chunk hold chunk_blocks items
    k_check_items<<<(n_items + 255) / 256, 256, 0, s>>>(MODE == MV_DIGEST ? nullptr : phys, n_items, c->NB, iw, (u32)std::min<u64>(c->cap_entries, 0xFFFFFFFFu),
                                                         ispos, (u32)std::min<u64>(staged_limit, 0xFFFFFFFFu), c->d_check);
    c->st.kernel_launches++;
  }
  if (c->mover == RC_MOVER_TMA) {
    const TmaVariant& v = kTma[c->tma_variant[MODE]];
    const u32 grid = std::min(n_items * c->G, c->tma_grid[MODE]);
    v.fn[MODE]<<<grid, tma_block(v), tma_smem(v), s>>>(c->pool, staging, phys, part, n_items, c->G, c->NB, (u32)c->page, iw, ispos, sw, sg);
  } else launch_ldg<MODE>(c, s, staging, phys, part, n_items, iw, ispos, sw, sg);
  c->st.kernel_launches++;
}

// ---- create / destroy ------------------------------------------------------------------------
extern "C" int rc_destroy(rc_ctx* c) {
  if (!c) return RC_ERR_INVALID;
  cudaDeviceSynchronize();
  auto F = [](void* p) { if (p) cudaFree(p); };
  auto FH = [](void* p) { if (p) cudaFreeHost(p); };
  F(c->d_used); F(c->d_ref); F(c->d_bt); F(c->d_dg); F(c->d_dg2); F(c->d_ring); F(c->d_evcount); F(c->d_bitmaps); F(c->d_up);
  F(c->d_counters); F(c->d_alloc); F(c->d_flip); F(c->d_posmax); F(c->d_gain); F(c->d_protmap);
  for (u32 r = 0; r < TP_MAX_RANKS; ++r) if (c->peer_ipc[r] && c->peer_mb[r]) cudaIpcCloseMemHandle(c->peer_mb[r]);
  F(c->d_mailbox); F(c->d_verd); F(c->d_gath); FH(c->h_verd);
  for (int i = 0; i < 4; ++i) { F(c->d_desc[i]); F(c->d_res[i]); F(c->d_off[i]); FH(c->h_desc[i]); FH(c->h_res[i]); }
  for (int i = 0; i < 3; ++i) {
    F(c->d_phys[i]); F(c->d_dtmp[i]); F(c->d_etmp[i]);
    if (c->ev_body_a[i]) cudaEventDestroy(c->ev_body_a[i]);
    if (c->ev_body_b[i]) cudaEventDestroy(c->ev_body_b[i]);
  }
  FH(c->h_up); FH(c->h_flip); FH(c->h_counters); FH(c->h_check); FH(c->h_evbuf); FH(c->h_dig); FH(c->h_dig2); FH(c->h_iw); FH(c->h_ispos); FH(c->h_hpos);
  F(c->d_iw); F(c->d_ispos); F(c->d_hpos);
  FH(c->h_store);
  for (int d = 0; d < 2; ++d) {
    for (auto p : c->staging[d]) F(p);
    for (auto p : c->part[d]) F(p);
    for (auto e : c->ev_free[d]) cudaEventDestroy(e);
    for (auto e : c->ev_ready[d]) cudaEventDestroy(e);
    if (c->ev_plan[d]) cudaEventDestroy(c->ev_plan[d]);
  }
  for (auto e : c->ev_pool) cudaEventDestroy(e);
  cudaStream_t* ss[5] = {&c->meta, &c->gather, &c->d2h, &c->scatter, &c->h2d};
  for (int i = 0; i < 5; ++i) if (c->own[i] && *ss[i]) cudaStreamDestroy(*ss[i]);
  if (c->util) cudaStreamDestroy(c->util);
  delete c;
  return RC_OK;
}

extern "C" int rc_create(const rc_config* cfg, rc_ctx** out) {
  if (!cfg || !out) return RC_ERR_INVALID;
  *out = nullptr;
  const u64 page = (u64)cfg->block_size * cfg->kv_heads * cfg->head_dim * cfg->elem_bytes;
  if (!cfg->layers || !cfg->pool_blocks || page == 0 || page % 4096 != 0 || page > (1ull << 30)) return RC_ERR_INVALID;
  if (cfg->elem_bytes != 1 && cfg->elem_bytes != 2) return RC_ERR_INVALID;
  if (cfg->block_size > 255 || !cfg->pool_dev || !cfg->fill_dev || ((uintptr_t)cfg->pool_dev & 255)) return RC_ERR_INVALID;
  if (!cfg->max_claims || !cfg->max_table_entries || !cfg->max_events || cfg->staging_chunks < 2) return RC_ERR_INVALID;
  const u64 blk = 2ull * cfg->layers * page;
  if (cfg->staging_chunk_bytes < blk || cfg->mover > RC_MOVER_TMA) return RC_ERR_INVALID;
  if (cfg->tp_ranks > TP_MAX_RANKS || (cfg->tp_ranks ? cfg->tp_rank >= cfg->tp_ranks : cfg->tp_rank != 0)) return RC_ERR_INVALID;
  if (cfg->tp_ranks > 1 && cfg->dedup) return RC_ERR_INVALID;        // the content-addressed store is not sharded
  if (cfg->layer_major > 1 || (cfg->layer_major && (cfg->dedup || cfg->direct_offload))) return RC_ERR_INVALID;
  if ((cfg->staging_chunk_bytes / blk) * (2ull * cfg->layers) > 0x7FFFFFFFull) return RC_ERR_INVALID;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return RC_ERR_CUDA;   // no device, no library
  rc_ctx* c = new rc_ctx();
  c->cfg = *cfg;
  c->page = page; c->blk = blk; c->G = 2 * cfg->layers; c->vpp = (u32)(page / 16); c->NB = cfg->pool_blocks;
  c->R = cfg->staging_chunks;
  c->chunk_blocks = cfg->staging_chunk_bytes / blk;
  c->host_blocks = cfg->host_store_bytes / blk;
  c->cap_entries = cfg->max_table_entries;
  c->desc_cap = 2ull * cfg->max_claims + 1024;
  c->pool = (u8*)cfg->pool_dev; c->fill = cfg->fill_dev;
  memset(&c->st, 0, sizeof(c->st));
  c->host_alloc.init(c->host_blocks); c->bt_alloc.init(c->cap_entries); c->dg_alloc.init(c->cap_entries);
  auto fail = [&](int code, const char* what, cudaError_t e) {
    fprintf(stderr, "librc: rc_create failed at %s: %s\n", what, e == cudaSuccess ? "" : cudaGetErrorString(e));
    rc_destroy(c);
    return code;
  };
#define CC(call, code) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return fail(code, #call, e_); } while (0)
  cudaDeviceProp prop;
  int dev = 0;
  CC(cudaGetDevice(&dev), RC_ERR_CUDA);
  CC(cudaGetDeviceProperties(&prop, dev), RC_ERR_CUDA);
  c->sms = prop.multiProcessorCount;
  void* given[5] = {cfg->stream_meta, cfg->stream_gather, cfg->stream_d2h, cfg->stream_scatter, cfg->stream_h2d};
  cudaStream_t* ss[5] = {&c->meta, &c->gather, &c->d2h, &c->scatter, &c->h2d};
  for (int i = 0; i < 5; ++i) {
    if (given[i]) *ss[i] = (cudaStream_t)given[i];
    else { CC(cudaStreamCreateWithFlags(ss[i], cudaStreamNonBlocking), RC_ERR_CUDA); c->own[i] = true; }
  }
  CC(cudaStreamCreateWithFlags(&c->util, cudaStreamNonBlocking), RC_ERR_CUDA);
  const u64 NB = c->NB, cap = c->cap_entries, dc = c->desc_cap;
  CC(cudaMalloc(&c->d_used, NB), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_ref, NB * 4), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_bt, cap * 4), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_dg, cap * 8), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_dg2, cap * 8), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_ring, (u64)cfg->max_events * sizeof(Event)), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_evcount, 8), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_bitmaps, (u64)c->accept_ctas * ((NB + 31) / 32) * 4), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_up, cap * 4), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_counters, 16), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_alloc, cap * 4), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_flip, dc * 8), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_posmax, NB * 4), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_gain, dc * 4), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_protmap, NB), RC_ERR_NOMEM);
  c->tp_ranks = cfg->tp_ranks ? cfg->tp_ranks : 1; c->tp_rank = cfg->tp_rank;
  c->mailbox_bytes = TP_MAX_RANKS * 8 + (u64)c->tp_ranks * dc * sizeof(TpVerdict);
  CC(cudaMalloc(&c->d_mailbox, c->mailbox_bytes), RC_ERR_NOMEM);
  CC(cudaMemset(c->d_mailbox, 0, c->mailbox_bytes), RC_ERR_CUDA);
  CC(cudaMalloc(&c->d_verd, dc * sizeof(TpVerdict)), RC_ERR_NOMEM);
  CC(cudaMalloc(&c->d_gath, (u64)c->tp_ranks * dc * sizeof(TpVerdict)), RC_ERR_NOMEM);
  CC(cudaHostAlloc(&c->h_verd, (u64)c->tp_ranks * dc * sizeof(TpVerdict), cudaHostAllocMapped), RC_ERR_NOMEM);
  c->peer_mb[c->tp_rank] = c->d_mailbox;
  CC(cudaMemset(c->d_used, 0, NB), RC_ERR_CUDA);
  CC(cudaMemset(c->d_ref, 0, NB * 4), RC_ERR_CUDA);
  CC(cudaMemset(c->d_evcount, 0, 8), RC_ERR_CUDA);
  CC(cudaMemset(c->d_bitmaps, 0, (u64)c->accept_ctas * ((NB + 31) / 32) * 4), RC_ERR_CUDA);
  for (int i = 0; i < 4; ++i) {
    CC(cudaMalloc(&c->d_desc[i], dc * sizeof(Desc)), RC_ERR_NOMEM);
    CC(cudaMalloc(&c->d_res[i], dc * sizeof(Res)), RC_ERR_NOMEM);
    CC(cudaMalloc(&c->d_off[i], (dc + 1) * 4), RC_ERR_NOMEM);
    CC(cudaHostAlloc(&c->h_desc[i], dc * sizeof(Desc), cudaHostAllocMapped), RC_ERR_NOMEM);
    CC(cudaHostAlloc(&c->h_res[i], dc * sizeof(Res), cudaHostAllocMapped), RC_ERR_NOMEM);
  }
  CC(cudaHostAlloc(&c->h_up, cap * 4, cudaHostAllocMapped), RC_ERR_NOMEM);
  CC(cudaHostAlloc(&c->h_flip, dc * 8, cudaHostAllocMapped), RC_ERR_NOMEM);
  CC(cudaHostAlloc(&c->h_counters, 16, cudaHostAllocMapped), RC_ERR_NOMEM);
  CC(cudaHostAlloc(&c->h_check, 4, cudaHostAllocMapped), RC_ERR_NOMEM);
  *c->h_check = 0;
  CC(cudaHostGetDevicePointer((void**)&c->d_check, c->h_check, 0), RC_ERR_CUDA);
  if (const char* e = getenv("RC_CHECK")) c->check = atoi(e) != 0;
  c->ev_bounce_cap = std::min<u64>(cfg->max_events, 1u << 16);
  CC(cudaHostAlloc(&c->h_evbuf, c->ev_bounce_cap * sizeof(Event), cudaHostAllocMapped), RC_ERR_NOMEM);
  c->dedup = cfg->dedup != 0;
  c->direct = cfg->direct_offload != 0 && !c->dedup;
  c->lm = cfg->layer_major != 0;
  if (c->direct) {
    CC(cudaHostAlloc(&c->h_hpos, cap * 4, cudaHostAllocMapped), RC_ERR_NOMEM);
    CC(cudaMalloc(&c->d_hpos, cap * 4), RC_ERR_NOMEM);
  }
  if (c->dedup) {
    CC(cudaHostAlloc(&c->h_dig, cap * 8, cudaHostAllocMapped), RC_ERR_NOMEM);
    CC(cudaHostAlloc(&c->h_dig2, cap * 8, cudaHostAllocMapped), RC_ERR_NOMEM);
    CC(cudaHostAlloc(&c->h_iw, cap * 4, cudaHostAllocMapped), RC_ERR_NOMEM);
    CC(cudaHostAlloc(&c->h_ispos, cap * 4, cudaHostAllocMapped), RC_ERR_NOMEM);
    CC(cudaMalloc(&c->d_iw, cap * 4), RC_ERR_NOMEM);
    CC(cudaMalloc(&c->d_ispos, cap * 4), RC_ERR_NOMEM);
  }
  for (int i = 0; i < 3; ++i) {
    CC(cudaMalloc(&c->d_phys[i], cap * 4), RC_ERR_NOMEM);
    CC(cudaMalloc(&c->d_dtmp[i], cap * 8), RC_ERR_NOMEM);
    CC(cudaMalloc(&c->d_etmp[i], cap * 8), RC_ERR_NOMEM);
    CC(cudaEventCreateWithFlags(&c->ev_body_a[i], cudaEventDisableTiming), RC_ERR_CUDA);
    CC(cudaEventCreateWithFlags(&c->ev_body_b[i], cudaEventDisableTiming), RC_ERR_CUDA);
  }
  for (int d = 0; d < 2; ++d) {
    c->staging[d].assign(c->R, nullptr); c->part[d].assign(c->R, nullptr);
    c->ev_free[d].assign(c->R, nullptr); c->ev_ready[d].assign(c->R, nullptr);
    c->slot_used[d].assign(c->R, false);
    for (u32 r = 0; r < c->R; ++r) {
      CC(cudaMalloc(&c->staging[d][r], c->chunk_blocks * blk), RC_ERR_NOMEM);
      CC(cudaMalloc(&c->part[d][r], c->chunk_blocks * c->G * WPC * 16), RC_ERR_NOMEM);
      CC(cudaEventCreateWithFlags(&c->ev_free[d][r], cudaEventDisableTiming), RC_ERR_CUDA);
      CC(cudaEventCreateWithFlags(&c->ev_ready[d][r], cudaEventDisableTiming), RC_ERR_CUDA);
    }
    CC(cudaEventCreateWithFlags(&c->ev_plan[d], cudaEventDisableTiming), RC_ERR_CUDA);
  }
  if (c->host_blocks) CC(cudaHostAlloc(&c->h_store, c->host_blocks * blk, cudaHostAllocMapped), RC_ERR_NOMEM);
  if (c->host_blocks && c->direct) CC(cudaHostGetDevicePointer((void**)&c->h_store_dev, c->h_store, 0), RC_ERR_CUDA);
  // launch geometry of the movers
  c->mover = cfg->mover == RC_MOVER_AUTO ? RC_MOVER_TMA : cfg->mover;
  if (c->mover == RC_MOVER_TMA) {
    // Measured on B200 with the mum fold (profiles/r02_mover_sweep.md): the fused movers want about 64 KiB of bulk
    // loads in flight per SM -- 8 KiB tiles x 4 stages x 2 CTAs/SM (variant 1) wins for 32 KiB and 16 KiB pages alike;
    // the read-only digest pass runs at twice the byte rate and wants two folding groups (variants 10 / 15).
    for (int m = 0; m < 3; ++m) {
      int want = page % 8192 == 0 ? 1 : 0;
      if (m == MV_DIGEST) want = page % 32768 == 0 ? 10 : (page % 16384 == 0 ? 15 : want);
      if (const char* e = getenv("RC_TMA_VARIANT")) want = atoi(e);
      if (m == MV_DIGEST) if (const char* e = getenv("RC_TMA_VARIANT_DIGEST")) want = atoi(e);
      if (want < 0 || want >= kTmaN || page % kTma[want].tile != 0) return fail(RC_ERR_INVALID, "RC_TMA_VARIANT", cudaSuccess);
      c->tma_variant[m] = want;
      const TmaVariant& v = kTma[want];
      int o = 0;
      CC(cudaFuncSetAttribute(v.fn[m], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tma_smem(v)), RC_ERR_CUDA);
      CC(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, v.fn[m], (int)tma_block(v), tma_smem(v)), RC_ERR_CUDA);
      o = std::max(1, std::min<int>(o, v.ctas_per_sm));
      c->tma_grid[m] = cfg->grid_ctas ? cfg->grid_ctas : c->sms * (u32)o;
    }
  }
  int occ = 0;
  CC(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_move_hash<MV_GATHER, 8>, LANES, 0), RC_ERR_CUDA);
  occ = std::max(1, std::min(occ, 2));
  c->grid = cfg->grid_ctas ? cfg->grid_ctas : c->sms * (u32)occ;
#undef CC
  *out = c;
  return RC_OK;
}

// ---- small helpers -----------------------------------------------------------------------------
static int ev_room(rc_ctx* c, u64 extra) {
  return (c->ev_emitted - c->ev_drained) + c->ev_reserved + extra <= c->cfg.max_events;
}
static int upload_desc(rc_ctx* c, int set, u32 n) {
  CK(to_dev(c, c->meta, c->d_desc[set], c->h_desc[set], (u64)n * sizeof(Desc)));
  return RC_OK;
}
static int fetch_res(rc_ctx* c, int set, u32 n) {
  CK(to_host(c, c->meta, c->h_res[set], c->d_res[set], (u64)n * sizeof(Res)));
  return RC_OK;
}
static int emit(rc_ctx* c, int set, u32 n, int mode, u64 request_id = 0) {
  k_emit<<<1, 256, 0, c->meta>>>(c->d_desc[set], c->d_res[set], n, mode, c->d_ring, c->cfg.max_events, c->d_evcount, request_id,
                                 c->tp_ranks > 1);
  CKL();
  c->st.kernel_launches++;
  return RC_OK;
}
#define GUARD()                                   \
  if (!c) return RC_ERR_INVALID;                  \
  if (c->poisoned) return RC_ERR_CUDA

static int mark(rc_ctx* c, u32 n, const u32* ids, int val) {
  GUARD();
  if (n && !ids) return RC_ERR_INVALID;
  for (u32 i = 0; i < n; ++i) if (ids[i] >= c->NB) return RC_ERR_INVALID;
  for (u32 s = 0; s < n; s += (u32)c->cap_entries) {
    const u32 m = (u32)std::min<u64>(n - s, c->cap_entries);
    memcpy(c->h_up, ids + s, (u64)m * 4);
    CK(to_dev(c, c->meta, c->d_up, c->h_up, (u64)m * 4));
    k_mark<<<(m + 255) / 256, 256, 0, c->meta>>>(c->d_up, m, c->d_used, c->d_ref, val);
    CKL();
    c->st.kernel_launches++;
    CK(cudaStreamSynchronize(c->meta));
  }
  return RC_OK;
}
// fill_dev[ids[i]] = vals[i] from HOST arrays, through the small-transfer path (no copy engine: an admission made while
// chunk copies are in flight does not wait behind them).  Ids are packed in front of the values in the upload buffer.
extern "C" int rc_set_fill(rc_ctx* c, uint32_t n, const uint32_t* ids, const uint8_t* vals) {
  GUARD();
  if (n && (!ids || !vals)) return RC_ERR_INVALID;
  for (u32 i = 0; i < n; ++i) if (ids[i] >= c->NB || vals[i] > c->cfg.block_size) return RC_ERR_INVALID;
  const u32 per = (u32)std::min<u64>(std::max<u64>(1, c->cap_entries * 4 / 5 - 1), 1u << 30);   // 4 B id + 1 B value per entry, values padded to 4 B
  for (u32 s = 0; s < n; s += per) {
    const u32 m = std::min(per, n - s), vb = (m + 3) & ~3u;
    memcpy(c->h_up, ids + s, (u64)m * 4);
    memcpy((u8*)(c->h_up + m), vals + s, m);
    CK(to_dev(c, c->meta, c->d_up, c->h_up, (u64)m * 4 + vb));
    k_fill_write<<<(m + 255) / 256, 256, 0, c->meta>>>(c->d_up, (const u8*)(c->d_up + m), m, c->fill);
    CKL();
    c->st.kernel_launches++;
    CK(cudaStreamSynchronize(c->meta));
  }
  return RC_OK;
}
extern "C" int rc_mark_used(rc_ctx* c, uint32_t n, const uint32_t* ids) { return mark(c, n, ids, 1); }
extern "C" int rc_mark_free(rc_ctx* c, uint32_t n, const uint32_t* ids) { return mark(c, n, ids, 0); }

// ---- a0 accept -----------------------------------------------------------------------------------
constexpr u64 NO_EXT = ~0ull;
static bool accept_shape_ok(rc_ctx* c, u64 id, u32 P, u32 N, u32 o0, u32 o1) {
  return id != 0 && P != 0 && N != 0 && N <= P && o1 >= o0 && o1 - o0 == ceil_div(P, c->cfg.block_size);
}
// One run of a batch (no id twice inside a run).  ext[k] = the table extent rc_accept reserved for entry k before the
// first run (NO_EXT for entries whose shape is invalid); an extent that ends up unused is given back here.
static int accept_run(rc_ctx* c, u32 n, const u64* id, const u32* P, const u32* N, const u32* bt_off, const u32* bt_ids,
                      int32_t* st, u64* ext) {
  Desc* hd = c->h_desc[2];
  std::vector<u32> cand;
  u64 up = 0;
  auto give_back = [&](u32 k) { if (ext[k] != NO_EXT) { c->bt_alloc.release(ext[k], bt_off[k + 1] - bt_off[k]); ext[k] = NO_EXT; } };
  for (u32 k = 0; k < n; ++k) {
    memset(&hd[k], 0, sizeof(Desc));
    hd[k].id = id[k];
    if (id[k] == 0) { st[k] = RC_ST_UNKNOWN_CLAIM; give_back(k); continue; }          // 0 is "no claim"
    if (c->claims.count(id[k])) { st[k] = RC_ST_DUPLICATE_ID; give_back(k); continue; } // duplicate ownership
    if (!accept_shape_ok(c, id[k], P[k], N[k], bt_off[k], bt_off[k + 1])) { st[k] = RC_ST_BAD_TABLE; give_back(k); continue; }
    const u32 nt = bt_off[k + 1] - bt_off[k];
    const u64 o = ext[k];
    hd[k].P = P[k]; hd[k].N = N[k]; hd[k].bt_off = (u32)o; hd[k].bt_len = nt; hd[k].flags = D_ELIG;
    hd[k].src_off = (u32)up;
    memcpy(c->h_up + up, bt_ids + bt_off[k], (u64)nt * 4);
    up += nt;
    cand.push_back(k);
    st[k] = -1;
  }
  if (cand.empty()) return RC_OK;
  int rc;
  if ((rc = upload_desc(c, 2, n))) return rc;
  CK(to_dev(c, c->meta, c->d_up, c->h_up, up * 4));
  k_accept<<<std::min<u32>(n, c->accept_ctas), 256, 0, c->meta>>>(c->d_desc[2], c->d_res[2], n, c->d_up, c->d_bt, c->d_used,
                                                                 c->d_ref, c->NB, c->d_bitmaps);
  CKL();
  c->st.kernel_launches++;
  if ((rc = emit(c, 2, n, EM_ACCEPT))) return rc;
  if ((rc = fetch_res(c, 2, n))) return rc;
  CK(cudaStreamSynchronize(c->meta));
  for (u32 k : cand) {
    if (c->h_res[2][k].flag & R_OK) {
      Claim cl;
      cl.id = id[k]; cl.state = RC_CS_ACCEPTED; cl.P = P[k]; cl.N = N[k]; cl.order = c->accept_seq++;
      cl.bt_off = hd[k].bt_off; cl.bt_len = hd[k].bt_len;
      c->claims.emplace(id[k], std::move(cl));
      c->ev_emitted++;
      st[k] = RC_ST_OK;
    } else {
      c->bt_alloc.release(hd[k].bt_off, hd[k].bt_len);
      st[k] = RC_ST_BAD_TABLE;
    }
    ext[k] = NO_EXT;
  }
  return RC_OK;
}

extern "C" int rc_accept(rc_ctx* c, uint32_t n, const uint64_t* id, const uint32_t* P, const uint32_t* N,
                         const uint32_t* bt_off, const uint32_t* bt_ids, int32_t* st) {
  GUARD();
  if (n == 0) return RC_OK;
  if (!id || !P || !N || !bt_off || !st || (bt_off[n] && !bt_ids)) return RC_ERR_INVALID;
  if (c->claims.size() + n > c->cfg.max_claims || !ev_room(c, n)) return RC_ERR_CAPACITY;
  // every table extent of the batch is reserved before the first run mutates anything, so RC_ERR_CAPACITY leaves no
  // claim accepted and no event emitted (rc.h: a negative return changes nothing)
  std::vector<u64> ext(n, NO_EXT);
  u64 per_run = 0;
  bool fits = true;
  for (u32 k = 0; k < n && fits; ++k) {
    if (!accept_shape_ok(c, id[k], P[k], N[k], bt_off[k], bt_off[k + 1])) continue;
    const u32 nt = bt_off[k + 1] - bt_off[k];
    per_run += nt;
    fits = per_run <= c->cap_entries && c->bt_alloc.alloc(nt, ext[k]);       // the upload buffer holds one run; a run <= the batch
    if (!fits) ext[k] = NO_EXT;
  }
  if (!fits) {
    for (u32 k = 0; k < n; ++k) if (ext[k] != NO_EXT) c->bt_alloc.release(ext[k], bt_off[k + 1] - bt_off[k]);
    return RC_ERR_CAPACITY;
  }
  // a run never holds the same id twice, so the runs reproduce one-by-one acceptance
  u32 s = 0;
  int rc = RC_OK;
  while (s < n && rc == RC_OK) {
    std::unordered_set<u64> seen;
    u32 e = s;
    while (e < n && e - s < c->desc_cap && (id[e] == 0 || seen.insert(id[e]).second)) ++e;
    rc = accept_run(c, e - s, id + s, P + s, N + s, bt_off + s, bt_ids, st + s, ext.data() + s);
    s = e;
  }
  for (u32 k = 0; k < n; ++k) if (ext[k] != NO_EXT) c->bt_alloc.release(ext[k], bt_off[k + 1] - bt_off[k]);   // CUDA error path
  return rc;
}

// ---- a1 materialize --------------------------------------------------------------------------------
extern "C" int rc_materialize(rc_ctx* c, uint32_t n, const uint64_t* id, int32_t* st) {
  GUARD();
  if (n == 0) return RC_OK;
  if (!id || !st || n > c->desc_cap) return RC_ERR_INVALID;
  if (!ev_room(c, n)) return RC_ERR_CAPACITY;
  Desc* hd = c->h_desc[2];
  std::unordered_map<u64, u32> first;
  std::vector<std::pair<u32, u32>> dups;
  std::vector<u32> cand;
  for (u32 k = 0; k < n; ++k) {
    memset(&hd[k], 0, sizeof(Desc));
    hd[k].id = id[k];
    auto it = c->claims.find(id[k]);
    if (it == c->claims.end()) { st[k] = RC_ST_UNKNOWN_CLAIM; continue; }   // post-hoc naming
    Claim& cl = it->second;
    if (cl.busy || cl.state != RC_CS_ACCEPTED) { st[k] = RC_ST_BAD_STATE; continue; }
    auto f = first.find(id[k]);
    if (f != first.end()) { dups.push_back({k, f->second}); continue; }
    first[id[k]] = k;
    hd[k].P = cl.P; hd[k].N = cl.N; hd[k].bt_off = cl.bt_off; hd[k].bt_len = cl.bt_len; hd[k].flags = D_ELIG;
    cand.push_back(k);
  }
  if (!cand.empty()) {
    int rc;
    if ((rc = upload_desc(c, 2, n))) return rc;
    k_pred<<<warps_grid(n), 256, 0, c->meta>>>(c->d_desc[2], c->d_res[2], n, c->d_bt, c->fill, c->cfg.block_size);
    CKL();
    c->st.kernel_launches++;
    if ((rc = emit(c, 2, n, EM_MATERIALIZE))) return rc;
    if ((rc = fetch_res(c, 2, n))) return rc;
    CK(cudaStreamSynchronize(c->meta));
    for (u32 k : cand) {
      const Res r = c->h_res[2][k];
      if (r.flag & R_OK) {
        Claim& cl = c->claims[id[k]];
        cl.M = r.val; cl.nb = ceil_div(r.val, c->cfg.block_size); cl.state = RC_CS_MATERIALIZED;
        c->ev_emitted++;
        st[k] = RC_ST_OK;
      } else st[k] = RC_ST_PRED_FALSE;
    }
  }
  for (auto& d : dups) st[d.first] = st[d.second] == RC_ST_OK ? RC_ST_BAD_STATE : RC_ST_PRED_FALSE;
  return RC_OK;
}

// ---- transfer engine helpers --------------------------------------------------------------------
// copies the host-store segments that intersect work positions [w0, w1) of a chunk
static int copy_chunk(rc_ctx* c, int dir, cudaStream_t s, u8* stg, u64 w0, u64 w1, const std::vector<Seg>& segs, size_t& si,
                      u64& bytes) {
  u8 *ha = nullptr, *da = nullptr; u64 len = 0;
  auto flush = [&]() -> cudaError_t {
    if (!len) return cudaSuccess;
    cudaError_t e = dir == 0 ? cudaMemcpyAsync(ha, da, len, cudaMemcpyDeviceToHost, s)
                             : cudaMemcpyAsync(da, ha, len, cudaMemcpyHostToDevice, s);
    bytes += len; len = 0;
    return e;
  };
  while (si < segs.size() && segs[si].w0 < w1) {
    const Seg& g = segs[si];
    const u64 a = std::max(g.w0, w0), b = std::min(g.w0 + g.n, w1);
    if (a < b) {
      u8* h = c->h_store + (g.hoff + (a - g.w0)) * c->blk;
      u8* d = stg + (a - w0) * c->blk;
      const u64 l = (b - a) * c->blk;
      if (len && h == ha + len && d == da + len) len += l;
      else { CK(flush()); ha = h; da = d; len = l; }
    }
    if (g.w0 + g.n <= w1) ++si; else break;
  }
  CK(flush());
  return RC_OK;
}

// Layer-major mode (rc.h rc_config.layer_major): a claim's host copy is [g][block i][page] -- all its blocks' page 0, then
// page 1, ... -- laid over its host-store extents in order, and a staging chunk of m items is [g][item][page].  The copies
// of a chunk are issued plane by plane, so within a chunk the bytes cross the link in layer order.
struct LmClaim { u64 w0; u32 nb; const std::vector<std::pair<u64, u64>>* host; };
static int copy_chunk_lm(rc_ctx* c, int dir, cudaStream_t s, u8* stg, u64 w0, u64 w1, const std::vector<LmClaim>& cls, size_t& ci,
                         u64& bytes) {
  const u64 m = w1 - w0, page = c->page;
  u8 *ha = nullptr, *da = nullptr; u64 len = 0;
  auto flush = [&]() -> cudaError_t {
    if (!len) return cudaSuccess;
    cudaError_t e = dir == 0 ? cudaMemcpyAsync(ha, da, len, cudaMemcpyDeviceToHost, s)
                             : cudaMemcpyAsync(da, ha, len, cudaMemcpyHostToDevice, s);
    bytes += len; len = 0;
    return e;
  };
  size_t last = ci;
  for (u32 g = 0; g < c->G; ++g) {
    for (size_t k = ci; k < cls.size() && cls[k].w0 < w1; ++k) {
      const LmClaim& q = cls[k];
      const u64 a = std::max(q.w0, w0), b = std::min(q.w0 + q.nb, w1);
      if (a >= b) continue;
      last = k;
      u64 v = ((u64)g * q.nb + (a - q.w0)) * page, left = (b - a) * page;        // run in the claim's host copy
      u8* d = stg + ((u64)g * m + (a - w0)) * page;
      u64 base = 0;                                                              // virtual offset of the extent
      for (auto& e : *q.host) {
        const u64 eb = e.second * c->blk;
        if (left && v < base + eb) {
          const u64 l = std::min(left, base + eb - v);
          u8* h = c->h_store + e.first * c->blk + (v - base);
          if (len && h == ha + len && d == da + len) len += l;
          else { CK(flush()); ha = h; da = d; len = l; }
          v += l; d += l; left -= l;
        }
        base += eb;
      }
    }
  }
  CK(flush());
  if (last < cls.size() && cls[last].w0 + cls[last].nb <= w1) ci = last + 1; else ci = last;   // first claim of the next chunk
  return RC_OK;
}

extern "C" int rc_wait(rc_ctx* c, int which);
// ---- a1-a4 offload ------------------------------------------------------------------------------------
static int offload_begin_dedup(rc_ctx* c, uint32_t n, const uint64_t* id, int32_t* st);
static int restore_begin_dedup(rc_ctx* c, uint32_t n, const uint64_t* id, int32_t* st);
static void dedup_drop(rc_ctx* c, Claim& cl);

// Chunk boundaries of an operation over T work positions: chunks of chunk_blocks items.  A restore cuts its LAST chunk
// in two: the scatter of the final piece is the one mover launch that no H2D copy hides (the link idles while it runs),
// so that piece is a quarter chunk -- 0.15 ms of scatter instead of 0.6 ms per operation, +1 % on a step of 2 GiB
// waves.  Not smaller: a launch of a sixteenth chunk runs at 0.6 of the rate of a full one (measured: scatter 0.926
// overall instead of 0.987).  An offload is not cut: its first gather delays a direction that runs ahead anyway.
static std::vector<std::pair<u64, u64>> plan_chunks(const rc_ctx* c, u64 T, bool short_last) {
  std::vector<std::pair<u64, u64>> ch;
  for (u64 w0 = 0; w0 < T; w0 += c->chunk_blocks) ch.push_back({w0, std::min(T, w0 + c->chunk_blocks)});
  const u64 tail = std::max<u64>(1, c->chunk_blocks / 4);
  if (short_last && !ch.empty()) {
    auto l = ch.back();
    if (l.second - l.first > 2 * tail) { ch.back().second = l.second - tail; ch.push_back({l.second - tail, l.second}); }
  }
  return ch;
}

// ---- offload slots ------------------------------------------------------------------------------------
// Up to OFF_DEPTH offloads may be open (begun, not yet completed by rc_wait(0)); they run back to back on the gather
// and d2h streams.  _begin enqueues a1-a3 and the chain; the a4 bookkeeping -- reference drop, OFFLOADED -- is enqueued
// on `meta` when rc_wait(0) completes the oldest open offload, so on `meta` it takes the place of that call.
constexpr int OFF_DEPTH = 2;
static inline int off_oi(int slot) { return slot ? 2 : 0; }      // op index: ops[], d_phys[], d_dtmp[], d_etmp[], ev_body_*[]
static inline int off_set(int slot) { return slot ? 3 : 0; }     // descriptor / result set
static int off_take_slot(const rc_ctx* c) {
  if (c->off_open >= OFF_DEPTH) return -1;
  return c->off_open == 0 ? 0 : (c->off_q[0] ^ 1);
}
// data movement of the offload in `slot` is enqueued: mark its end on both streams and open it
static int offload_opened(rc_ctx* c, int slot, u32 n_served) {
  const int oi = off_oi(slot);
  CK(cudaEventRecord(c->ev_body_a[oi], c->gather));
  CK(cudaEventRecord(c->ev_body_b[oi], c->d2h));
  c->ev_reserved += n_served;
  c->ops[oi].active = true;
  c->off_q[c->off_open++] = slot;
  return RC_OK;
}

extern "C" int rc_offload_begin(rc_ctx* c, uint32_t n, const uint64_t* id, int32_t* st) {
  GUARD();
  if (c->dedup) return offload_begin_dedup(c, n, id, st);
  const int slot_o = off_take_slot(c);
  if (slot_o < 0 || (c->direct && c->off_open)) return RC_ERR_BUSY;   // the direct mover's index buffer is single
  if (n == 0) return RC_OK;
  if (!id || !st || n > c->desc_cap) return RC_ERR_INVALID;
  if (!ev_room(c, n)) return RC_ERR_CAPACITY;
  const int oi = off_oi(slot_o), set = off_set(slot_o);
  Op& op = c->ops[oi];
  Desc* hd = c->h_desc[set];
  op.cl.assign(n, nullptr);
  std::vector<Seg> segs;
  std::vector<LmClaim> lmc;                               // layer-major mode: served claims by work position
  std::vector<u32> served;
  bool full = false;
  u64 T = 0;
  std::vector<std::pair<u32, u32>> old_dg;                 // per served claim: the digest extent recorded by an earlier cycle
  auto rollback = [&]() {                                  // a negative return changes no claim (rc.h)
    for (size_t j = 0; j < served.size(); ++j) {
      Claim& cl = *op.cl[served[j]];
      for (auto& e : cl.host) c->host_alloc.release(e.first, e.second);
      cl.host.clear();
      c->host_used -= (u64)cl.nb * c->blk;
      c->dg_alloc.release(cl.dg_off, cl.dg_len);
      cl.dg_off = old_dg[j].first; cl.dg_len = old_dg[j].second;
      cl.busy = false;
    }
  };
  for (u32 k = 0; k < n; ++k) {
    memset(&hd[k], 0, sizeof(Desc));
    hd[k].id = id[k];
    auto it = c->claims.find(id[k]);
    if (it == c->claims.end()) { st[k] = RC_ST_UNKNOWN_CLAIM; continue; }
    Claim& cl = it->second;
    // no claim-less entry point exists: "ordinary offload without claim" cannot produce an outcome
    if (cl.busy || (cl.state != RC_CS_MATERIALIZED && cl.state != RC_CS_RESIDENT_AGAIN)) { st[k] = RC_ST_BAD_STATE; continue; }
    if (full || c->host_used + (u64)cl.nb * c->blk > c->cfg.host_store_bytes) { full = true; st[k] = RC_ST_NO_HOST_SPACE; continue; }
    u64 dgo;                                               // new extent first; the old one goes once the batch is admitted
    if (T + cl.nb > c->cap_entries || !c->dg_alloc.alloc(cl.nb, dgo)) { rollback(); return RC_ERR_CAPACITY; }
    old_dg.push_back({cl.dg_off, cl.dg_len});
    cl.dg_off = (u32)dgo; cl.dg_len = cl.nb;
    cl.host.clear();
    // host space is granted by count in _begin order (a restore in flight still holds its bytes: it gives them
    // back when rc_wait(1) completes it)
    c->host_alloc.alloc_split(cl.nb, cl.host);
    c->host_used += (u64)cl.nb * c->blk;
    cl.busy = true;
    op.cl[k] = &cl;
    served.push_back(k);
    hd[k].P = cl.P; hd[k].N = cl.N; hd[k].M = cl.M; hd[k].nb = cl.nb; hd[k].bt_off = cl.bt_off; hd[k].bt_len = cl.bt_len;
    hd[k].dg_off = cl.dg_off; hd[k].flags = D_ELIG;
    u64 w = T;
    for (auto& e : cl.host) { segs.push_back({w, e.second, e.first}); w += e.second; }
    if (c->lm) lmc.push_back({T, cl.nb, &cl.host});
    T += cl.nb;
    st[k] = -1;
  }
  if (served.empty()) return RC_OK;
  for (auto& od : old_dg) if (od.second) c->dg_alloc.release(od.first, od.second);
  op.n = n; op.status = st; op.blocks = T; op.copy_bytes = 0; op.launches = 0;
  int rc;
  // The head (offsets, compaction) only reads tables that completed calls wrote, so it runs on the gather stream;
  // nothing of an offload touches `meta` before rc_wait(0).
  CK(to_dev(c, c->gather, c->d_desc[set], c->h_desc[set], (u64)n * sizeof(Desc)));
  k_offsets<<<1, 1024, 0, c->gather>>>(c->d_desc[set], n, c->d_off[set]);
  CKL();
  k_worklist<<<warps_grid(n), 256, 0, c->gather>>>(c->d_desc[set], c->d_res[set], n, c->d_off[set], c->d_bt, nullptr, c->d_phys[oi], 0);
  CKL();
  c->st.kernel_launches += 2;
  size_t si = 0, li = 0;
  for (const auto& ch : plan_chunks(c, T, false)) {
    const u64 w0 = ch.first, w1 = ch.second;
    const u32 slot = (u32)(c->chunk_seq[0]++ % c->R), m = (u32)(w1 - w0);      // the ring runs on across operations
    if (c->direct) {
      // the mover's destination is the claim's place in the mapped pinned store: the bulk stores of the gather
      // kernel cross the link themselves (item -> host block through the same indirection the dedup restore uses)
      while (si < segs.size() && segs[si].w0 < w1) {
        const Seg& g = segs[si];
        for (u64 w = std::max(g.w0, w0); w < std::min(g.w0 + g.n, w1); ++w) c->h_hpos[w] = (u32)(g.hoff + (w - g.w0));
        if (g.w0 + g.n <= w1) ++si; else break;
      }
      CK(to_dev(c, c->gather, c->d_hpos + w0, c->h_hpos + w0, (u64)m * 4));
      cudaEvent_t t0 = get_event(c), t1 = get_event(c);
      CK(cudaEventRecord(t0, c->gather));
      launch_move<MV_GATHER>(c, c->gather, c->h_store_dev, c->d_phys[oi] + w0, c->part[0][slot], m, nullptr, c->d_hpos + w0);
      CKL();
      CK(cudaEventRecord(t1, c->gather));
      op.t_copy.push_back({t0, t1});                       // the kernel IS the transfer
      op.copy_bytes += (u64)m * c->blk;
      k_block_digest<<<warps_grid(m), 256, 0, c->gather>>>(c->part[0][slot], nullptr, c->d_dtmp[oi] + w0, c->d_etmp[oi] + w0, m, c->G, nullptr);
      CKL();
      c->st.kernel_launches++;
      continue;
    }
    if (c->slot_used[0][slot]) CK(cudaStreamWaitEvent(c->gather, c->ev_free[0][slot], 0));
    cudaEvent_t t0 = get_event(c), t1 = get_event(c);
    CK(cudaEventRecord(t0, c->gather));
    launch_move<MV_GATHER>(c, c->gather, c->staging[0][slot], c->d_phys[oi] + w0, c->part[0][slot], m, nullptr, nullptr, c->lm);
    CKL();
    CK(cudaEventRecord(t1, c->gather));
    op.t_kernel.push_back({t0, t1});
    op.launches++;
    k_block_digest<<<warps_grid(m), 256, 0, c->gather>>>(c->part[0][slot], nullptr, c->d_dtmp[oi] + w0, c->d_etmp[oi] + w0, m, c->G, nullptr);
    CKL();
    c->st.kernel_launches++;
    CK(cudaEventRecord(c->ev_ready[0][slot], c->gather));
    CK(cudaStreamWaitEvent(c->d2h, c->ev_ready[0][slot], 0));
    cudaEvent_t c0 = get_event(c), c1 = get_event(c);
    CK(cudaEventRecord(c0, c->d2h));
    if ((rc = c->lm ? copy_chunk_lm(c, 0, c->d2h, c->staging[0][slot], w0, w1, lmc, li, op.copy_bytes)
                    : copy_chunk(c, 0, c->d2h, c->staging[0][slot], w0, w1, segs, si, op.copy_bytes))) return rc;
    CK(cudaEventRecord(c1, c->d2h));
    op.t_copy.push_back({c0, c1});
    CK(cudaEventRecord(c->ev_free[0][slot], c->d2h));
    c->slot_used[0][slot] = true;
  }
  k_chain<<<warps_grid(n), 256, 0, c->gather>>>(c->d_desc[set], c->d_res[set], n, c->d_off[set], c->d_dtmp[oi], c->d_etmp[oi], c->d_dg, c->d_dg2);
  CKL();
  c->st.kernel_launches++;
  return offload_opened(c, slot_o, (u32)served.size());
}

static int collect_times(rc_ctx* c, Op& op, float& ms_k, float& ms_c) {
  static const bool trace = getenv("RC_TRACE_LAUNCHES") != nullptr;      // diagnostics: per-launch device times on stderr
  if (trace) {
    const int dir = &op == &c->ops[1];
    for (auto& p : op.t_kernel) { float ms = 0; cudaEventElapsedTime(&ms, p.first, p.second); fprintf(stderr, "librc trace: %s kernel %.4f ms\n", dir ? "scatter" : "gather", ms); }
    for (auto& p : op.t_copy) { float ms = 0; cudaEventElapsedTime(&ms, p.first, p.second); fprintf(stderr, "librc trace: %s copy %.4f ms\n", dir ? "h2d" : "d2h", ms); }
  }
  for (auto& p : op.t_kernel) { float ms = 0; CK(cudaEventElapsedTime(&ms, p.first, p.second)); ms_k += ms; c->ev_pool.push_back(p.first); c->ev_pool.push_back(p.second); }
  for (auto& p : op.t_copy) { float ms = 0; CK(cudaEventElapsedTime(&ms, p.first, p.second)); ms_c += ms; c->ev_pool.push_back(p.first); c->ev_pool.push_back(p.second); }
  op.t_kernel.clear(); op.t_copy.clear();
  return RC_OK;
}

// Completes the oldest open offload: a4 on `meta` (after the transfer: "offloaded" follows the finished copy),
// then the host-side claim records.
static int check_flag(rc_ctx* c) {                         // after the operation's streams have been waited for
  if (c->check && *c->h_check) { c->poisoned = true; c->cuda_err = "RC_CHECK: a work item of a mover launch was out of range"; return RC_ERR_CUDA; }
  return RC_OK;
}

static int wait_offload(rc_ctx* c) {
  if (!c->off_open) return RC_OK;
  const int slot = c->off_q[0], oi = off_oi(slot), set = off_set(slot);
  Op& op = c->ops[oi];
  const u32 n = op.n;
  int rc;
  CK(cudaStreamWaitEvent(c->meta, c->ev_body_a[oi], 0));
  CK(cudaStreamWaitEvent(c->meta, c->ev_body_b[oi], 0));
  k_unref<<<warps_grid(n), 256, 0, c->meta>>>(c->d_desc[set], n, c->d_bt, c->d_used, c->d_ref);
  CKL();
  c->st.kernel_launches++;
  if ((rc = emit(c, set, n, EM_OFFLOAD))) return rc;
  CK(to_host(c, c->meta, c->h_res[set], c->d_res[set], (u64)n * sizeof(Res)));
  CK(cudaStreamSynchronize(c->meta));
  if ((rc = check_flag(c))) return rc;
  op.active = false;
  c->off_q[0] = c->off_q[1]; --c->off_open;
  u64 served = 0;
  for (u32 k = 0; k < op.n; ++k) {
    Claim* cl = op.cl[k];
    if (!cl) continue;
    cl->chain = c->h_res[set][k].chain;
    cl->state = RC_CS_OFFLOADED;
    c->bt_alloc.release(cl->bt_off, cl->bt_len);
    cl->bt_len = 0;
    cl->busy = false;
    op.status[k] = RC_ST_OK;
    ++served;
  }
  c->ev_reserved -= served; c->ev_emitted += served;
  c->st.claims_offloaded += served; c->st.bytes_d2h += op.copy_bytes;
  c->st.gather_launches += op.launches; c->st.gather_blocks += op.blocks;
  return collect_times(c, op, c->st.ms_gather, c->st.ms_d2h);
}

// ---- a5-a8 restore ---------------------------------------------------------------------------------------
// the restore's data movement is enqueued: mark its end and open it.  Its verdicts and outcome records (a7-a8) are
// enqueued on `meta` by rc_wait(1), so on `meta` they take the place of that call; the plan (a5) took place at _begin.
static int restore_opened(rc_ctx* c, u32 n_served) {
  Op& op = c->ops[1];
  CK(cudaEventRecord(c->ev_body_a[1], c->scatter));
  op.request_id = c->request_id; op.tp = c->tp_split; op.tail = false;
  c->ev_reserved += 4ull * n_served;
  op.active = true;
  return RC_OK;
}
// a7 on `meta`, after the data movement: digests and chain compared, verdict; then a8 -- or, in the TP split form, the
// local verdict records published (to the host for the all-gather path, into the peers' mailboxes for the NVLink path):
// there the merged verdict is applied and the outcomes are emitted by rc_tp_restore_commit.
static int restore_tail(rc_ctx* c) {
  Op& op = c->ops[1];
  if (op.tail) return RC_OK;
  const u32 n = op.n;
  int rc;
  CK(cudaStreamWaitEvent(c->meta, c->ev_body_a[1], 0));
  k_verify<<<warps_grid(n), 256, 0, c->meta>>>(c->d_desc[1], c->d_res[1], n, c->d_off[1], c->d_dtmp[1], c->d_etmp[1], c->d_dg, c->d_dg2, c->d_bt,
                                               c->d_used, c->d_ref, c->fill, c->cfg.block_size, op.tp ? 0 : 1);
  CKL();
  c->st.kernel_launches++;
  if (op.tp) {
    k_tp_verdicts<<<(n + 255) / 256, 256, 0, c->meta>>>(c->d_res[1], n, c->d_verd);
    CKL();
    TpPeers peers;
    for (u32 r = 0; r < TP_MAX_RANKS; ++r) {
      u8* mb = r < c->tp_ranks ? c->peer_mb[r] : nullptr;
      peers.flag[r] = (u64*)mb;
      peers.rec[r] = mb ? (TpVerdict*)(mb + TP_MAX_RANKS * 8) : nullptr;
    }
    k_tp_push<<<1, 1024, 0, c->meta>>>(c->d_verd, n, peers, c->tp_ranks, c->tp_rank, (u32)c->desc_cap, c->tp_epoch);
    CKL();
    c->st.kernel_launches += 2;
    CK(to_host(c, c->meta, c->h_verd, c->d_verd, (u64)n * sizeof(TpVerdict)));
  } else {
    if ((rc = emit(c, 1, n, EM_RESTORE, op.request_id))) return rc;
    CK(to_host(c, c->meta, c->h_res[1], c->d_res[1], (u64)n * sizeof(Res)));
  }
  op.tail = true;
  return RC_OK;
}

extern "C" int rc_restore_begin(rc_ctx* c, uint32_t n, const uint64_t* id, int32_t* st) {
  GUARD();
  if (c->tp_pending) return RC_ERR_BUSY;                   // a split (TP) restore is waiting for its commit
  if (c->dedup) return restore_begin_dedup(c, n, id, st);
  Op& op = c->ops[1];
  if (op.active) return RC_ERR_BUSY;
  if (n == 0) return RC_OK;
  if (!id || !st || n > c->desc_cap) return RC_ERR_INVALID;
  Desc* hd = c->h_desc[1];
  op.cl.assign(n, nullptr);
  std::vector<u32> elig;
  std::unordered_set<u64> seen;
  u64 Te = 0;
  auto rollback = [&]() { for (u32 k : elig) c->bt_alloc.release(hd[k].bt_off, hd[k].nb); };
  for (u32 k = 0; k < n; ++k) {
    memset(&hd[k], 0, sizeof(Desc));
    hd[k].id = id[k];
    auto it = c->claims.find(id[k]);
    if (it == c->claims.end()) { st[k] = RC_ST_UNKNOWN_CLAIM; continue; }
    Claim& cl = it->second;
    // restore-after-use and double restore are not OFFLOADED any more
    if (cl.busy || cl.state != RC_CS_OFFLOADED || !seen.insert(id[k]).second) { st[k] = RC_ST_BAD_STATE; continue; }
    u64 o;
    if (Te + cl.nb > c->cap_entries || !c->bt_alloc.alloc(cl.nb, o)) { rollback(); return RC_ERR_CAPACITY; }
    hd[k].chain = cl.chain; hd[k].P = cl.P; hd[k].N = cl.N; hd[k].M = cl.M; hd[k].nb = cl.nb;
    hd[k].bt_off = (u32)o; hd[k].bt_len = cl.nb; hd[k].dg_off = cl.dg_off; hd[k].flags = D_ELIG; hd[k].pad = cl.policy;
    op.cl[k] = &cl;
    elig.push_back(k);
    Te += cl.nb;
    st[k] = -1;
  }
  if (elig.empty()) return RC_OK;
  if (!ev_room(c, 4ull * elig.size())) { rollback(); for (u32 k : elig) st[k] = RC_ST_BAD_STATE; return RC_ERR_CAPACITY; }
  int rc;
  if ((rc = upload_desc(c, 1, n))) return rc;
  k_restore_plan<<<1, 1024, 0, c->meta>>>(c->d_desc[1], c->d_res[1], n, c->d_off[1], c->d_used, c->d_ref, c->NB, c->d_alloc,
                                          c->d_counters);
  CKL();
  c->st.kernel_launches++;
  CK(to_host(c, c->meta, c->h_res[1], c->d_res[1], (u64)n * sizeof(Res)));
  CK(cudaStreamSynchronize(c->meta));                    // the grant (which claims are served) is needed to plan the copies
  std::vector<Seg> segs;
  std::vector<LmClaim> lmc;
  std::vector<std::pair<u64, u64>> flips;                // (work position, byte in block = g*page + byte in page)
  u64 T = 0;
  u32 n_served = 0;
  bool reupload = false;
  for (u32 k : elig) {
    Claim& cl = *op.cl[k];
    if (!(c->h_res[1][k].flag & R_SERVED)) {
      c->bt_alloc.release(hd[k].bt_off, hd[k].nb);
      op.cl[k] = nullptr;
      st[k] = RC_ST_NO_FREE_BLOCKS;
      continue;
    }
    ++n_served;
    cl.busy = true;
    // fault decision: the first armed entry naming exactly this claim, one-shot.  Entries naming any
    // other id never fire for it (wrong-claim / unclaimed failures are not claim outcomes: P:L25)
    rc_fault flt{0, 0, 0};
    for (size_t f = 0; f < c->faults.size(); ++f)
      if (c->faults[f].claim_id == id[k]) { flt = c->faults[f]; c->faults.erase(c->faults.begin() + f); break; }
    if (flt.kind == RC_FAULT_XFER_ERROR) { hd[k].flags |= D_XFER; reupload = true; }
    else {
      if (flt.kind == RC_FAULT_BITFLIP) {
        const u64 pos = flt.param % ((u64)cl.nb * c->blk);   // a byte of the claim's host copy, in ITS layout
        if (c->lm) {
          const u64 plane = (u64)cl.nb * c->page, g = pos / plane, r = pos % plane;
          flips.push_back({T + r / c->page, g * c->page + r % c->page});
        } else flips.push_back({T + pos / c->blk, pos % c->blk});
      }
      u64 w = T;
      for (auto& e : cl.host) { segs.push_back({w, e.second, e.first}); w += e.second; }
      if (c->lm) lmc.push_back({T, cl.nb, &cl.host});
    }
    T += cl.nb;
  }
  if (n_served == 0) return RC_OK;
  if (c->fault_flags & RC_FAULT_ALLOW_UNCLAIMED)          // a counter, never an outcome
    for (size_t f = 0; f < c->faults.size();)
      if (c->faults[f].claim_id == 0) { c->st.generic_failures++; c->faults.erase(c->faults.begin() + f); } else ++f;
  op.n = n; op.status = st; op.blocks = T; op.copy_bytes = 0; op.launches = 0;
  if (reupload && (rc = upload_desc(c, 1, n))) return rc;
  k_worklist<<<warps_grid(n), 256, 0, c->meta>>>(c->d_desc[1], c->d_res[1], n, c->d_off[1], c->d_bt, c->d_alloc, c->d_phys[1], 1);
  CKL();
  c->st.kernel_launches++;
  CK(cudaEventRecord(c->ev_plan[1], c->meta));
  CK(cudaStreamWaitEvent(c->scatter, c->ev_plan[1], 0));
  std::sort(flips.begin(), flips.end());
  size_t si = 0, fi = 0, li = 0;
  u64 flip_base = 0;
  for (const auto& ch : plan_chunks(c, T, true)) {
    const u64 w0 = ch.first, w1 = ch.second;
    const u32 slot = (u32)(c->chunk_seq[1]++ % c->R), m = (u32)(w1 - w0);
    if (c->slot_used[1][slot]) CK(cudaStreamWaitEvent(c->h2d, c->ev_free[1][slot], 0));
    cudaEvent_t c0 = get_event(c), c1 = get_event(c);
    CK(cudaEventRecord(c0, c->h2d));
    if ((rc = c->lm ? copy_chunk_lm(c, 1, c->h2d, c->staging[1][slot], w0, w1, lmc, li, op.copy_bytes)
                    : copy_chunk(c, 1, c->h2d, c->staging[1][slot], w0, w1, segs, si, op.copy_bytes))) return rc;
    CK(cudaEventRecord(c1, c->h2d));
    op.t_copy.push_back({c0, c1});
    CK(cudaEventRecord(c->ev_ready[1][slot], c->h2d));
    CK(cudaStreamWaitEvent(c->scatter, c->ev_ready[1][slot], 0));
    u32 nf = 0;
    while (fi < flips.size() && flips[fi].first < w1) {  // injected corruption of the staged copy (host bytes stay intact)
      const u64 fw = flips[fi].first - w0, fb = flips[fi].second;          // item in the chunk, byte in the block
      c->h_flip[flip_base + nf++] = c->lm ? ((fb / c->page) * m + fw) * c->page + fb % c->page : fw * c->blk + fb;
      ++fi;
    }
    if (nf) {
      CK(to_dev(c, c->scatter, c->d_flip + flip_base, c->h_flip + flip_base, (u64)nf * 8));
      k_bitflip<<<(nf + 63) / 64, 64, 0, c->scatter>>>(c->staging[1][slot], c->d_flip + flip_base, nf);
      CKL();
      c->st.kernel_launches++;
      flip_base += nf;
    }
    cudaEvent_t t0 = get_event(c), t1 = get_event(c);
    CK(cudaEventRecord(t0, c->scatter));
    launch_move<MV_SCATTER>(c, c->scatter, c->staging[1][slot], c->d_phys[1] + w0, c->part[1][slot], m, nullptr, nullptr, c->lm);
    CKL();
    CK(cudaEventRecord(t1, c->scatter));
    op.t_kernel.push_back({t0, t1});
    op.launches++;
    k_block_digest<<<warps_grid(m), 256, 0, c->scatter>>>(c->part[1][slot], c->d_phys[1] + w0, c->d_dtmp[1] + w0, c->d_etmp[1] + w0, m, c->G, nullptr);
    CKL();
    c->st.kernel_launches++;
    CK(cudaEventRecord(c->ev_free[1][slot], c->scatter));
    c->slot_used[1][slot] = true;
  }
  return restore_opened(c, n_served);
}

static int wait_restore(rc_ctx* c) {
  Op& op = c->ops[1];
  if (!op.active) return RC_OK;
  int rc;
  if ((rc = restore_tail(c))) return rc;
  CK(cudaStreamSynchronize(c->meta));
  if ((rc = check_flag(c))) return rc;
  op.active = false;
  const Desc* hd = c->h_desc[1];
  for (u32 k = 0; k < op.n; ++k) {
    Claim* cl = op.cl[k];
    if (!cl) continue;
    const Res r = c->h_res[1][k];
    // the host copy ends with the restore (success or not): space and extents go back now
    if (c->dedup) dedup_drop(c, *cl);
    else c->host_used -= (u64)cl->nb * c->blk;
    for (auto& e : cl->host) c->host_alloc.release(e.first, e.second);
    cl->host.clear();
    cl->busy = false;
    c->ev_reserved -= 4;
    if (r.flag & R_OK) {
      cl->state = RC_CS_RESIDENT_AGAIN; cl->bt_off = hd[k].bt_off; cl->bt_len = cl->nb;
      c->ev_emitted += 2; c->st.claims_restored++;
      op.status[k] = RC_ST_OK;
    } else {
      c->bt_alloc.release(hd[k].bt_off, cl->nb);
      if (cl->dg_len) { c->dg_alloc.release(cl->dg_off, cl->dg_len); cl->dg_len = 0; }
      cl->bt_len = 0;
      cl->state = cl->policy == POL_DEMOTE ? RC_CS_DEMOTED : (cl->policy == POL_EXPIRE ? RC_CS_EXPIRED : RC_CS_REFUSED);   // terminal
      c->ev_emitted += 4; c->st.claims_refused++;
      op.status[k] = RC_ST_RESTORE_FAILED;
    }
  }
  c->st.bytes_h2d += op.copy_bytes;
  c->st.scatter_launches += op.launches; c->st.scatter_blocks += op.blocks;
  return collect_times(c, op, c->st.ms_scatter, c->st.ms_h2d);
}

extern "C" int rc_wait(rc_ctx* c, int which) {
  GUARD();
  if (which == 0) return wait_offload(c);
  if (which == 1) return c->tp_pending ? RC_ERR_BUSY : wait_restore(c);   // a split restore ends with rc_tp_restore_commit
  return RC_ERR_INVALID;
}
extern "C" int rc_offload(rc_ctx* c, uint32_t n, const uint64_t* id, int32_t* st) {
  int rc = rc_offload_begin(c, n, id, st);
  while (rc == RC_OK && c->off_open) rc = wait_offload(c);     // open offloads complete in _begin order, this one last
  return rc;
}
extern "C" int rc_test(rc_ctx* c, int which, int* done) {
  GUARD();
  if (!done || which < 0 || which > 1) return RC_ERR_INVALID;
  *done = 1;
  cudaError_t e = cudaSuccess;
  if (which == 0 && c->off_open) {                             // the transfer of the oldest open offload
    const int oi = off_oi(c->off_q[0]);
    e = cudaEventQuery(c->ev_body_a[oi]);
    if (e == cudaSuccess) e = cudaEventQuery(c->ev_body_b[oi]);
  } else if (which == 1 && c->ops[1].active) e = cudaEventQuery(c->ev_body_a[1]);   // H2D + scatter + digests
  if (e == cudaErrorNotReady) { *done = 0; return RC_OK; }
  CK(e);
  return RC_OK;
}
extern "C" int rc_restore(rc_ctx* c, uint32_t n, const uint64_t* id, int32_t* st) {
  const int rc = rc_restore_begin(c, n, id, st);
  return rc ? rc : wait_restore(c);
}

// ---- NEXT-4: TP-sharded restore (rc.h; DESIGN.md 8 / R24) ---------------------------------------------------------
extern "C" int rc_tp_restore_verify(rc_ctx* c, uint32_t n, const uint64_t* id, int32_t* st, rc_tp_verdict* local) {
  GUARD();
  if (c->dedup || c->tp_pending || (n && (!id || !st || !local))) return RC_ERR_INVALID;
  if (c->ops[1].active) return RC_ERR_BUSY;
  ++c->tp_epoch;
  c->tp_split = true;
  const int rc = rc_restore_begin(c, n, id, st);
  c->tp_split = false;
  if (rc) { --c->tp_epoch; return rc; }
  for (u32 k = 0; k < n; ++k) { local[k].flags = 0; local[k].bad = 0xFFFFFFFFu; }
  Op& op = c->ops[1];
  if (op.active) {
    int rt;
    if ((rt = restore_tail(c))) return rt;               // local verdicts, published
    CK(cudaStreamSynchronize(c->meta));
    memcpy(local, c->h_verd, (u64)n * sizeof(TpVerdict));
    for (u32 k = 0; k < n; ++k) if (op.cl[k]) st[k] = -1;            // pending: decided by the commit
  } else {
    // nothing was served: this rank still publishes its (empty) records so that the peers' commits see its epoch
    TpPeers peers;
    for (u32 r = 0; r < TP_MAX_RANKS; ++r) {
      u8* mb = r < c->tp_ranks ? c->peer_mb[r] : nullptr;
      peers.flag[r] = (u64*)mb;
      peers.rec[r] = mb ? (TpVerdict*)(mb + TP_MAX_RANKS * 8) : nullptr;
    }
    if (n) {
      memcpy(c->h_verd, local, (u64)n * sizeof(TpVerdict));
      CK(to_dev(c, c->meta, c->d_verd, c->h_verd, (u64)n * sizeof(TpVerdict)));
    }
    k_tp_push<<<1, 1024, 0, c->meta>>>(c->d_verd, n, peers, c->tp_ranks, c->tp_rank, (u32)c->desc_cap, c->tp_epoch);
    CKL();
    c->st.kernel_launches++;
    CK(cudaStreamSynchronize(c->meta));
  }
  c->tp_pending = true; c->tp_n = n;
  return RC_OK;
}

extern "C" int rc_tp_restore_commit(rc_ctx* c, uint32_t n, uint32_t ranks, const rc_tp_verdict* gathered, int32_t* st) {
  GUARD();
  if (!c->tp_pending || n != c->tp_n || ranks != c->tp_ranks || (n && !st)) return RC_ERR_INVALID;
  Op& op = c->ops[1];
  const TpVerdict* src = nullptr;
  u32 stride = 0;
  CK(cudaMemsetAsync(c->d_counters, 0, 16, c->meta));
  if (gathered) {                                          // all-gather path: [ranks][n] records from the caller
    memcpy(c->h_verd, gathered, (u64)ranks * n * sizeof(TpVerdict));
    if (n) CK(to_dev(c, c->meta, c->d_gath, c->h_verd, (u64)ranks * n * sizeof(TpVerdict)));
    src = c->d_gath; stride = n;
  } else {                                                 // NVLink path: the peers wrote into this rank's mailbox
    k_tp_ready<<<1, 32, 0, c->meta>>>((const u64*)c->d_mailbox, ranks, c->tp_epoch, c->d_counters);
    CKL();
    c->st.kernel_launches++;
    CK(to_host(c, c->meta, c->h_counters, c->d_counters, 16));
    CK(cudaStreamSynchronize(c->meta));
    if (c->h_counters[0]) return RC_ERR_BUSY;              // some peer has not published this epoch yet: barrier first
    src = (const TpVerdict*)(c->d_mailbox + TP_MAX_RANKS * 8); stride = (u32)c->desc_cap;
  }
  if (!op.active) {                                        // nothing was served here; the peers must agree
    if (n && gathered) for (u64 i = 0; i < (u64)ranks * n; ++i) if (gathered[i].flags & TV_SERVED) return RC_ERR_INVALID;
    c->tp_pending = false;
    return RC_OK;
  }
  k_tp_merge<<<(n + 255) / 256, 256, 0, c->meta>>>(c->d_res[1], n, src, stride, ranks, c->d_counters + 1);
  CKL();
  c->st.kernel_launches++;
  CK(to_host(c, c->meta, c->h_counters, c->d_counters, 16));
  CK(cudaStreamSynchronize(c->meta));
  if (c->h_counters[1]) return RC_ERR_INVALID;             // a rank disagrees on which claims were served: nothing applied
  k_tp_apply<<<warps_grid(n), 256, 0, c->meta>>>(c->d_desc[1], c->d_res[1], n, c->d_bt, c->d_used, c->d_ref, c->fill,
                                                 c->cfg.block_size);
  CKL();
  c->st.kernel_launches++;
  int rc;
  if ((rc = emit(c, 1, n, EM_RESTORE, 0))) return rc;
  CK(to_host(c, c->meta, c->h_res[1], c->d_res[1], (u64)n * sizeof(Res)));
  op.status = st;
  c->tp_pending = false;
  return wait_restore(c);
}

extern "C" int rc_tp_mailbox(rc_ctx* c, void** dev, uint64_t* bytes) {
  GUARD();
  if (!dev || !bytes) return RC_ERR_INVALID;
  *dev = c->d_mailbox; *bytes = c->mailbox_bytes;
  return RC_OK;
}
extern "C" int rc_tp_set_peer(rc_ctx* c, uint32_t rank, void* mailbox_dev) {
  GUARD();
  if (rank >= c->tp_ranks || rank == c->tp_rank) return RC_ERR_INVALID;
  if (c->peer_ipc[rank] && c->peer_mb[rank]) { cudaIpcCloseMemHandle(c->peer_mb[rank]); c->peer_ipc[rank] = false; }
  c->peer_mb[rank] = (u8*)mailbox_dev;
  return RC_OK;
}
extern "C" int rc_tp_ipc_handle(rc_ctx* c, void* handle64) {
  GUARD();
  if (!handle64) return RC_ERR_INVALID;
  cudaIpcMemHandle_t h;
  CK(cudaIpcGetMemHandle(&h, c->d_mailbox));
  static_assert(sizeof(h) == 64, "CUDA IPC handles are 64 bytes");
  memcpy(handle64, &h, 64);
  return RC_OK;
}
extern "C" int rc_tp_open_peer(rc_ctx* c, uint32_t rank, const void* handle64) {
  GUARD();
  if (rank >= c->tp_ranks || rank == c->tp_rank || !handle64) return RC_ERR_INVALID;
  cudaIpcMemHandle_t h;
  memcpy(&h, handle64, 64);
  void* p = nullptr;
  CK(cudaIpcOpenMemHandle(&p, h, cudaIpcMemLazyEnablePeerAccess));
  if (c->peer_ipc[rank] && c->peer_mb[rank]) cudaIpcCloseMemHandle(c->peer_mb[rank]);
  c->peer_mb[rank] = (u8*)p; c->peer_ipc[rank] = true;
  return RC_OK;
}

#include "rc_dedup.inl"

// NEXT-3: one reuse request naming several claims; refusal carries exactly the failed subset (rc.h)
extern "C" int rc_restore_request_begin(rc_ctx* c, uint64_t request_id, uint32_t n, const uint64_t* id, int32_t* st) {
  GUARD();
  if (request_id == 0) return RC_ERR_INVALID;
  c->request_id = request_id;
  const int rc = rc_restore_begin(c, n, id, st);
  c->request_id = 0;
  return rc;
}
extern "C" int rc_restore_request(rc_ctx* c, uint64_t request_id, uint32_t n, const uint64_t* id, int32_t* st) {
  const int rc = rc_restore_request_begin(c, request_id, n, id, st);
  return rc ? rc : wait_restore(c);
}
extern "C" int rc_set_policy(rc_ctx* c, uint32_t n, const uint64_t* id, const uint32_t* policy) {
  GUARD();
  if (n && (!id || !policy)) return RC_ERR_INVALID;
  for (u32 k = 0; k < n; ++k) if (!c->claims.count(id[k]) || policy[k] > RC_POLICY_EXPIRE) return RC_ERR_INVALID;
  for (u32 k = 0; k < n; ++k) c->claims[id[k]].policy = policy[k];
  return RC_OK;
}

// ---- NEXT-3: allocator-side protection (rc.h, R23) -------------------------------------------------
extern "C" int rc_protect(rc_ctx* c, uint32_t n, const uint64_t* id, const uint32_t* on) {
  GUARD();
  if (n && (!id || !on)) return RC_ERR_INVALID;
  for (u32 k = 0; k < n; ++k) {
    auto it = c->claims.find(id[k]);
    if (it == c->claims.end() || on[k] > 1 || it->second.state >= RC_CS_REFUSED) return RC_ERR_INVALID;
  }
  for (u32 k = 0; k < n; ++k) c->claims[id[k]].protect = on[k];
  return RC_OK;
}

// live claims that hold a table, in victim order: unprotected first, then protected, acceptance order inside each
static void victim_list(rc_ctx* c, std::vector<Claim*>& list, u32& U) {
  std::vector<Claim*> grp[2];
  for (auto& kv : c->claims) {
    Claim& cl = kv.second;
    if (cl.bt_len && (cl.state == RC_CS_ACCEPTED || cl.state == RC_CS_MATERIALIZED || cl.state == RC_CS_RESIDENT_AGAIN))
      grp[cl.protect ? 1 : 0].push_back(&cl);
  }
  for (auto& g : grp) std::sort(g.begin(), g.end(), [](const Claim* a, const Claim* b) { return a->order < b->order; });
  list = grp[0];
  U = (u32)list.size();
  list.insert(list.end(), grp[1].begin(), grp[1].end());
}
static void fill_desc(Desc& d, const Claim& cl, u32 flags) {
  memset(&d, 0, sizeof(Desc));
  d.id = cl.id; d.P = cl.P; d.N = cl.N; d.M = cl.M; d.nb = cl.nb; d.bt_off = cl.bt_off; d.bt_len = cl.bt_len; d.flags = flags;
}

extern "C" int rc_make_room(rc_ctx* c, uint64_t request_id, uint32_t need, int32_t* status, uint64_t* ids, uint32_t cap,
                            uint32_t* n_ids) {
  GUARD();
  if (request_id == 0 || !status || !n_ids || (cap && !ids)) return RC_ERR_INVALID;
  if (c->off_open || c->ops[1].active) return RC_ERR_BUSY;
  *n_ids = 0;
  std::vector<Claim*> list;
  u32 U = 0;
  victim_list(c, list, U);
  const u32 n = (u32)list.size();
  if (n > c->desc_cap || !ev_room(c, n)) return RC_ERR_CAPACITY;
  Desc* hd = c->h_desc[2];
  for (u32 k = 0; k < n; ++k) fill_desc(hd[k], *list[k], D_ELIG | (list[k]->protect ? (u32)D_PROT : 0u));
  int rc;
  if (n) {
    if ((rc = upload_desc(c, 2, n))) return rc;
    CK(cudaMemsetAsync(c->d_posmax, 0, (u64)c->NB * 4, c->meta));
    k_vic_posmax<<<warps_grid(n), 256, 0, c->meta>>>(c->d_desc[2], n, c->d_bt, c->d_posmax);
    CKL();
    k_vic_gain<<<warps_grid(n), 256, 0, c->meta>>>(c->d_desc[2], n, c->d_bt, c->d_posmax, c->d_gain);
    CKL();
    c->st.kernel_launches += 2;
  }
  k_vic_decide<<<1, 1024, 0, c->meta>>>(c->d_gain, n, U, need, c->d_used, c->NB, c->d_counters);
  CKL();
  c->st.kernel_launches++;
  CK(to_host(c, c->meta, c->h_counters, c->d_counters, 16));
  CK(cudaStreamSynchronize(c->meta));
  const u32 oc = c->h_counters[0], lo = c->h_counters[1], hi = c->h_counters[2];
  if (oc == VO_FITS) { *status = RC_ST_OK; return RC_OK; }
  if (oc == VO_NOFREE) { *status = RC_ST_NO_FREE_BLOCKS; return RC_OK; }
  const u32 m = hi - lo;
  for (u32 k = 0; k < m; ++k) {
    fill_desc(hd[k], *list[lo + k], D_ELIG);
    if (*n_ids < cap) ids[*n_ids] = list[lo + k]->id;
    ++*n_ids;
  }
  if ((rc = upload_desc(c, 2, m))) return rc;
  if (oc == VO_EVICT) {
    // ordered release: DEMOTED is on the stream before the references are dropped (claim_demoted_before_loss)
    if ((rc = emit(c, 2, m, EM_DEMOTE, request_id))) return rc;
    k_unref<<<warps_grid(m), 256, 0, c->meta>>>(c->d_desc[2], m, c->d_bt, c->d_used, c->d_ref);
    CKL();
    c->st.kernel_launches++;
    CK(cudaStreamSynchronize(c->meta));
    for (u32 k = 0; k < m; ++k) {
      Claim& cl = *list[k];
      c->bt_alloc.release(cl.bt_off, cl.bt_len);
      cl.bt_len = 0;
      cl.state = RC_CS_DEMOTED;
    }
    *status = RC_ST_OK;
  } else {                                                 // nothing is evicted; the request is refused, naming the blockers
    if ((rc = emit(c, 2, m, EM_CONFLICT, request_id))) return rc;
    CK(cudaStreamSynchronize(c->meta));
    *status = RC_ST_PROTECTED_CONFLICT;
  }
  c->ev_emitted += m;
  return RC_OK;
}

extern "C" int rc_protected_map(rc_ctx* c, uint8_t* prot) {
  GUARD();
  if (!prot) return RC_ERR_INVALID;
  if (c->off_open || c->ops[1].active) return RC_ERR_BUSY;
  std::vector<Claim*> list;
  u32 U = 0;
  victim_list(c, list, U);
  const u32 n = (u32)list.size();
  if (n > c->desc_cap) return RC_ERR_CAPACITY;
  Desc* hd = c->h_desc[2];
  for (u32 k = 0; k < n; ++k) fill_desc(hd[k], *list[k], D_ELIG | (list[k]->protect ? (u32)D_PROT : 0u));
  CK(cudaMemsetAsync(c->d_protmap, 0, c->NB, c->meta));
  if (n) {
    int rc;
    if ((rc = upload_desc(c, 2, n))) return rc;
    k_prot_map<<<warps_grid(n), 256, 0, c->meta>>>(c->d_desc[2], n, c->d_bt, c->d_protmap);
    CKL();
    c->st.kernel_launches++;
  }
  CK(cudaMemcpyAsync(prot, c->d_protmap, c->NB, cudaMemcpyDeviceToHost, c->meta));
  CK(cudaStreamSynchronize(c->meta));
  return RC_OK;
}

// ---- outcomes, faults, release -----------------------------------------------------------------------------
extern "C" int rc_outcomes(rc_ctx* c, rc_event* buf, uint64_t cap, uint64_t* n_out) {
  GUARD();
  if (!n_out || (cap && !buf)) return RC_ERR_INVALID;
  const u64 m = std::min<u64>(cap, c->ev_emitted - c->ev_drained), E = c->cfg.max_events;
  // the records come back through a mapped pinned bounce buffer (small transfers: no copy engine), then to the caller
  u64 done = 0;
  while (done < m) {
    u64 part = std::min<u64>(m - done, c->ev_bounce_cap), got = 0;
    while (got < part) {
      const u64 at = (c->ev_drained + done + got) % E, l = std::min(part - got, E - at);
      CK(to_host(c, c->util, c->h_evbuf + got, c->d_ring + at, l * sizeof(Event)));
      got += l;
    }
    CK(cudaStreamSynchronize(c->util));
    memcpy(buf + done, c->h_evbuf, part * sizeof(Event));
    done += part;
  }
  c->ev_drained += m;
  *n_out = m;
  return RC_OK;
}

extern "C" int rc_set_faults(rc_ctx* c, uint32_t n, const rc_fault* f, uint32_t flags) {
  GUARD();
  if (n && !f) return RC_ERR_INVALID;
  for (u32 i = 0; i < n; ++i) {
    if (f[i].kind != RC_FAULT_XFER_ERROR && f[i].kind != RC_FAULT_BITFLIP) return RC_ERR_INVALID;
    if (f[i].claim_id == 0 && !(flags & RC_FAULT_ALLOW_UNCLAIMED)) return RC_ERR_INVALID;   // separate flag
  }
  c->faults.assign(f, f + n);
  c->fault_flags = flags;
  return RC_OK;
}

extern "C" int rc_release(rc_ctx* c, uint32_t n, const uint64_t* id, int32_t* st) {
  GUARD();
  if (n == 0) return RC_OK;
  if (!id || !st || n > c->desc_cap) return RC_ERR_INVALID;
  Desc* hd = c->h_desc[2];
  bool any = false;
  for (u32 k = 0; k < n; ++k) {
    memset(&hd[k], 0, sizeof(Desc));
    auto it = c->claims.find(id[k]);
    if (it == c->claims.end()) { st[k] = RC_ST_UNKNOWN_CLAIM; continue; }
    Claim& cl = it->second;
    if (cl.busy) { st[k] = RC_ST_BAD_STATE; continue; }
    if (cl.bt_len) {
      hd[k].bt_off = cl.bt_off; hd[k].bt_len = cl.bt_len; hd[k].flags = D_ELIG; any = true;
      c->bt_alloc.release(cl.bt_off, cl.bt_len);
    }
    if (cl.dg_len) c->dg_alloc.release(cl.dg_off, cl.dg_len);
    for (auto& e : cl.host) c->host_alloc.release(e.first, e.second);
    if (!cl.host.empty()) c->host_used -= (u64)cl.nb * c->blk;
    if (!cl.hkeys.empty()) dedup_drop(c, cl);
    c->claims.erase(it);
    st[k] = RC_ST_OK;
  }
  if (any) {
    int rc;
    if ((rc = upload_desc(c, 2, n))) return rc;
    k_unref<<<warps_grid(n), 256, 0, c->meta>>>(c->d_desc[2], n, c->d_bt, c->d_used, c->d_ref);
    CKL();
    c->st.kernel_launches++;
    CK(cudaStreamSynchronize(c->meta));
  }
  return RC_OK;
}

// ---- introspection -------------------------------------------------------------------------------------------
extern "C" int rc_claim_info(rc_ctx* c, uint64_t id, rc_claim_info_t* o) {
  GUARD();
  auto it = c->claims.find(id);
  if (it == c->claims.end() || !o) return RC_ERR_INVALID;
  const Claim& cl = it->second;
  o->claim_id = id; o->chain = cl.chain; o->host_bytes = (cl.host.empty() && cl.hslots.empty()) ? 0 : (u64)cl.nb * c->blk;
  o->state = cl.state; o->P = cl.P; o->N = cl.N; o->M = cl.M; o->nb = cl.nb; o->n_table = cl.bt_len;
  return RC_OK;
}
extern "C" int rc_claim_blocks(rc_ctx* c, uint64_t id, uint32_t* ids, uint32_t cap, uint32_t* n) {
  GUARD();
  auto it = c->claims.find(id);
  if (it == c->claims.end() || !n) return RC_ERR_INVALID;
  const Claim& cl = it->second;
  *n = cl.bt_len;
  const u32 m = std::min(cap, cl.bt_len);
  if (m && ids) {
    CK(cudaMemcpyAsync(ids, c->d_bt + cl.bt_off, (u64)m * 4, cudaMemcpyDeviceToHost, c->util));
    CK(cudaStreamSynchronize(c->util));
  }
  return RC_OK;
}
extern "C" int rc_claim_digests(rc_ctx* c, uint64_t id, uint64_t* d, uint64_t* e, uint32_t cap, uint32_t* n) {
  GUARD();
  auto it = c->claims.find(id);
  if (it == c->claims.end() || !n) return RC_ERR_INVALID;
  const Claim& cl = it->second;
  *n = cl.dg_len;
  const u32 m = std::min(cap, cl.dg_len);
  if (m && d) {
    CK(cudaMemcpyAsync(d, c->d_dg + cl.dg_off, (u64)m * 8, cudaMemcpyDeviceToHost, c->util));
    if (e) CK(cudaMemcpyAsync(e, c->d_dg2 + cl.dg_off, (u64)m * 8, cudaMemcpyDeviceToHost, c->util));
    CK(cudaStreamSynchronize(c->util));
  }
  return RC_OK;
}
extern "C" int rc_host_read(rc_ctx* c, uint64_t id, void* dst, uint64_t cap, uint64_t* bytes) {
  GUARD();
  auto it = c->claims.find(id);
  if (it == c->claims.end() || !bytes) return RC_ERR_INVALID;
  const Claim& cl = it->second;
  if (cl.busy && cl.state != RC_CS_OFFLOADED) return RC_ERR_BUSY;   // its offload is in flight: the host copy is not complete yet
  *bytes = (cl.host.empty() && cl.hslots.empty()) ? 0 : (u64)cl.nb * c->blk;
  if (dst && cap >= *bytes && *bytes) {
    u8* o = (u8*)dst;
    for (u32 sl : cl.hslots) { memcpy(o, c->h_store + (u64)sl * c->blk, c->blk); o += c->blk; }
    for (auto& e : cl.host) { memcpy(o, c->h_store + e.first * c->blk, e.second * c->blk); o += e.second * c->blk; }
  }
  return RC_OK;
}
extern "C" int rc_host_store(rc_ctx* c, uint64_t id, uint32_t block, const void** p, uint64_t* contiguous_bytes) {
  GUARD();
  if (c->lm) return RC_ERR_INVALID;                      // layer-major: a block is not contiguous in the host copy (rc_host_read)
  auto it = c->claims.find(id);
  if (it == c->claims.end() || !p || !contiguous_bytes) return RC_ERR_INVALID;
  const Claim& cl = it->second;
  if (cl.busy) return RC_ERR_BUSY;                         // an in-flight offload is still writing it
  *p = nullptr; *contiguous_bytes = 0;
  if (!cl.hslots.empty()) {                                // dedup store: one slot per block
    if (block >= cl.hslots.size()) return RC_ERR_INVALID;
    u64 run = 1;
    while (block + run < cl.hslots.size() && cl.hslots[block + run] == cl.hslots[block] + run) ++run;
    *p = c->h_store + (u64)cl.hslots[block] * c->blk; *contiguous_bytes = run * c->blk;
    return RC_OK;
  }
  u64 at = 0;
  for (auto& e : cl.host) {
    if (block < at + e.second) {
      *p = c->h_store + (e.first + (block - at)) * c->blk; *contiguous_bytes = (at + e.second - block) * c->blk;
      return RC_OK;
    }
    at += e.second;
  }
  return RC_ERR_INVALID;                                   // the claim holds no host bytes, or fewer blocks
}
extern "C" int rc_sync(rc_ctx* c) {
  GUARD();
  int rc = RC_OK;
  while (c->off_open) if ((rc = wait_offload(c))) return rc;
  if ((rc = wait_restore(c))) return rc;
  cudaStream_t ss[6] = {c->meta, c->gather, c->d2h, c->scatter, c->h2d, c->util};
  for (cudaStream_t s : ss) CK(cudaStreamSynchronize(s));
  return RC_OK;
}
extern "C" int rc_pool_state(rc_ctx* c, uint8_t* used, uint32_t* ref) {
  GUARD();
  if (used) CK(cudaMemcpyAsync(used, c->d_used, c->NB, cudaMemcpyDeviceToHost, c->util));
  if (ref) CK(cudaMemcpyAsync(ref, c->d_ref, (u64)c->NB * 4, cudaMemcpyDeviceToHost, c->util));
  CK(cudaStreamSynchronize(c->util));
  return RC_OK;
}
extern "C" int rc_stats_get(rc_ctx* c, rc_stats* o) {
  GUARD();
  if (!o) return RC_ERR_INVALID;
  std::vector<u8> used(c->NB);
  CK(cudaMemcpyAsync(used.data(), c->d_used, c->NB, cudaMemcpyDeviceToHost, c->util));
  CK(cudaStreamSynchronize(c->util));
  u64 fr = 0;
  for (u8 u : used) fr += !u;
  c->st.host_used_bytes = c->host_used; c->st.free_blocks = fr; c->st.events_emitted = c->ev_emitted;
  *o = c->st;
  return RC_OK;
}
extern "C" int rc_stats_reset(rc_ctx* c) {
  GUARD();
  const u64 g = c->st.generic_failures;
  memset(&c->st, 0, sizeof(c->st));
  c->st.generic_failures = g;
  return RC_OK;
}

// ---- measurement helpers -----------------------------------------------------------------------------------------
extern "C" int rc_measure_link(rc_ctx* c, uint64_t bytes, int direction, int reps, double* gbs) {
  GUARD();
  if (!gbs || direction < 0 || direction > 2 || reps < 1) return RC_ERR_INVALID;
  if (c->off_open || c->ops[1].active) return RC_ERR_BUSY;
  if (c->host_used != 0 || !c->store.empty()) return RC_ERR_BUSY;   // the measurement writes over the pinned store: only while it holds no claim bytes
  const u64 hs = c->host_blocks * c->blk, cs = c->chunk_blocks * c->blk;
  const u64 hmax = direction == 2 ? hs / 2 : hs;
  bytes = std::min(bytes, std::min(hmax, cs));
  if (bytes == 0) return RC_ERR_INVALID;
  cudaEvent_t a0 = get_event(c), a1 = get_event(c), b0 = get_event(c), b1 = get_event(c);
  double best = 0;
  for (int r = 0; r < reps; ++r) {
    CK(cudaDeviceSynchronize());
    float ma = 0, mb = 0;
    if (direction == 0 || direction == 2) {
      CK(cudaEventRecord(a0, c->d2h));
      CK(cudaMemcpyAsync(c->h_store, c->staging[0][0], bytes, cudaMemcpyDeviceToHost, c->d2h));
      CK(cudaEventRecord(a1, c->d2h));
    }
    if (direction == 1 || direction == 2) {
      CK(cudaEventRecord(b0, c->h2d));
      CK(cudaMemcpyAsync(c->staging[1][0], c->h_store + (direction == 2 ? hs / 2 : 0), bytes, cudaMemcpyHostToDevice, c->h2d));
      CK(cudaEventRecord(b1, c->h2d));
    }
    CK(cudaDeviceSynchronize());
    if (direction != 1) CK(cudaEventElapsedTime(&ma, a0, a1));
    if (direction != 0) CK(cudaEventElapsedTime(&mb, b0, b1));
    const double ms = std::max(ma, mb), g = (direction == 2 ? 2.0 : 1.0) * bytes / (ms * 1e6);
    best = std::max(best, g);
  }
  c->ev_pool.insert(c->ev_pool.end(), {a0, a1, b0, b1});
  *gbs = best;
  return RC_OK;
}

extern "C" int rc_digest_blocks(rc_ctx* c, const void* src, uint32_t n_blocks, uint64_t* digests, uint64_t* digests2,
                                float* ms_out) {
  GUARD();
  if (!src || ((uintptr_t)src & 15) || n_blocks > c->cap_entries) return RC_ERR_INVALID;
  if (c->off_open) return RC_ERR_BUSY;
  cudaEvent_t t0 = get_event(c), t1 = get_event(c);
  float total = 0;
  for (u64 w0 = 0; w0 < n_blocks; w0 += c->chunk_blocks) {
    const u32 m = (u32)std::min<u64>(c->chunk_blocks, n_blocks - w0);
    CK(cudaEventRecord(t0, c->gather));
    launch_move<MV_DIGEST>(c, c->gather, (u8*)src + w0 * c->blk, nullptr, c->part[0][0], m);
    CKL();
    CK(cudaEventRecord(t1, c->gather));
    k_block_digest<<<warps_grid(m), 256, 0, c->gather>>>(c->part[0][0], nullptr, c->d_dtmp[0] + w0, c->d_etmp[0] + w0, m, c->G, nullptr);
    CKL();
    CK(cudaStreamSynchronize(c->gather));
    float ms = 0;
    CK(cudaEventElapsedTime(&ms, t0, t1));
    total += ms;
  }
  if (n_blocks && (digests || digests2)) {
    if (digests) CK(cudaMemcpyAsync(digests, c->d_dtmp[0], (u64)n_blocks * 8, cudaMemcpyDeviceToHost, c->gather));
    if (digests2) CK(cudaMemcpyAsync(digests2, c->d_etmp[0], (u64)n_blocks * 8, cudaMemcpyDeviceToHost, c->gather));
    CK(cudaStreamSynchronize(c->gather));
  }
  c->ev_pool.push_back(t0); c->ev_pool.push_back(t1);
  if (ms_out) *ms_out = total;
  return RC_OK;
}

// ---- NEXT-1: trace validator ----------------------------------------------------------------------------------------
extern "C" int rc_validate_trace(const rc_event* events, uint64_t n, rc_trace_report* rep, rc_trace_claim* claims, uint64_t cap) {
  using namespace rct;
  if (!rep || (n && !events) || n > (1ull << 30)) return RC_ERR_INVALID;   // the claim table is 2n slots rounded up, in u32
  memset(rep, 0, sizeof(*rep));
  rep->first_bad_index = NO_BAD; rep->n_events = n; rep->ok = 1;
  if (n == 0) return RC_OK;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return RC_ERR_CUDA;
  u64 slots64 = 1024;
  while (slots64 < 2 * n) slots64 <<= 1;
  const u32 slots = (u32)slots64;                          // <= 2^31 by the bound on n
  Event* d_ev = nullptr; u64* d_keys = nullptr; u32 *d_count = nullptr, *d_base = nullptr, *d_dense = nullptr, *d_fill = nullptr;
  u32 *d_slot = nullptr, *d_bucket = nullptr, *d_cur = nullptr, *d_bsum = nullptr; unsigned long long* d_bad = nullptr; ClaimOut* d_out = nullptr;
  cudaStream_t st = nullptr; cudaEvent_t e0 = nullptr, e1 = nullptr, e2 = nullptr, e3 = nullptr;
  int rc = RC_OK;
  std::vector<ClaimOut> host_out;
#define TV(call) do { if ((call) != cudaSuccess) { rc = RC_ERR_CUDA; goto done; } } while (0)
  TV(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
  TV(cudaEventCreate(&e0)); TV(cudaEventCreate(&e1)); TV(cudaEventCreate(&e2)); TV(cudaEventCreate(&e3));
  TV(cudaMalloc(&d_ev, n * sizeof(Event))); TV(cudaMalloc(&d_keys, (u64)slots * 8)); TV(cudaMalloc(&d_count, (u64)slots * 4));
  TV(cudaMalloc(&d_base, (u64)slots * 4)); TV(cudaMalloc(&d_dense, (u64)slots * 4)); TV(cudaMalloc(&d_fill, (u64)slots * 4));
  TV(cudaMalloc(&d_slot, n * 4)); TV(cudaMalloc(&d_bucket, n * 4)); TV(cudaMalloc(&d_cur, 8)); TV(cudaMalloc(&d_bad, 8));
  TV(cudaMalloc(&d_out, n * sizeof(ClaimOut)));
  TV(cudaEventRecord(e0, st));
  TV(cudaMemcpyAsync(d_ev, events, n * sizeof(Event), cudaMemcpyHostToDevice, st));
  TV(cudaMemsetAsync(d_keys, 0, (u64)slots * 8, st)); TV(cudaMemsetAsync(d_count, 0, (u64)slots * 4, st));
  TV(cudaMemsetAsync(d_fill, 0, (u64)slots * 4, st)); TV(cudaMemsetAsync(d_cur, 0, 8, st));
  TV(cudaMemsetAsync(d_bad, 0xFF, 8, st));
  TV(cudaEventRecord(e1, st));
  tv_insert<<<(u32)((n + 255) / 256), 256, 0, st>>>((const Event*)d_ev, n, d_keys, d_count, slots - 1, d_slot, d_bad);
  tv_alloc<<<(slots + 255) / 256, 256, 0, st>>>(d_count, slots, d_base, d_dense, d_cur);
  tv_scatter<<<(u32)((n + 255) / 256), 256, 0, st>>>(n, d_slot, d_base, d_fill, d_bucket);
  {                                                        // request-level refusal runs (cross-claim rule)
    const u32 nbk = (u32)((n + 1023) / 1024);
    TV(cudaMalloc(&d_bsum, (u64)nbk * 4));
    tv_delta_sum<<<nbk, 1024, 0, st>>>((const Event*)d_ev, n, d_bsum);
    tv_scan_bsum<<<1, 1024, 0, st>>>(d_bsum, nbk);
    tv_groups<<<nbk, 1024, 0, st>>>((const Event*)d_ev, n, d_bsum, d_bad);
  }
  tv_walk<<<(slots + 127) / 128, 128, 0, st>>>((const Event*)d_ev, d_keys, d_count, slots, d_base, d_dense, d_bucket, d_out, d_bad);
  TV(cudaGetLastError());
  TV(cudaEventRecord(e2, st));
  {
    u32 cur[2]; unsigned long long bad;
    TV(cudaMemcpyAsync(cur, d_cur, 8, cudaMemcpyDeviceToHost, st));
    TV(cudaMemcpyAsync(&bad, d_bad, 8, cudaMemcpyDeviceToHost, st));
    TV(cudaStreamSynchronize(st));
    rep->n_claims = cur[1]; rep->first_bad_index = bad; rep->ok = bad == NO_BAD;
    host_out.resize(cur[1]);
    if (cur[1]) TV(cudaMemcpyAsync(host_out.data(), d_out, (u64)cur[1] * sizeof(ClaimOut), cudaMemcpyDeviceToHost, st));
    TV(cudaEventRecord(e3, st));
    TV(cudaStreamSynchronize(st));
    for (u64 k = 0; k < host_out.size(); ++k) {
      if (!rep->ok) host_out[k].gates = 0;                // the gates presuppose a valid stream
      rep->n_failure_gate += (host_out[k].gates & G_FAILURE) != 0;
      rep->n_observation_gate += (host_out[k].gates & G_OBSERVATION) != 0;
      if (claims && k < cap) memcpy(&claims[k], &host_out[k], sizeof(ClaimOut));
    }
    TV(cudaEventElapsedTime(&rep->ms_kernels, e1, e2));
    TV(cudaEventElapsedTime(&rep->ms_total, e0, e3));
  }
done:
#undef TV
  cudaFree(d_ev); cudaFree(d_keys); cudaFree(d_count); cudaFree(d_base); cudaFree(d_dense); cudaFree(d_fill);
  cudaFree(d_slot); cudaFree(d_bucket); cudaFree(d_cur); cudaFree(d_bad); cudaFree(d_out); cudaFree(d_bsum);
  if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1); if (e2) cudaEventDestroy(e2); if (e3) cudaEventDestroy(e3);
  if (st) cudaStreamDestroy(st);
  return rc;
}

extern "C" const char* rc_strerror(int err) {
  switch (err) {
    case RC_OK: return "ok";
    case RC_ERR_INVALID: return "invalid argument";
    case RC_ERR_CUDA: return "CUDA error (context poisoned) or no CUDA device";
    case RC_ERR_NOMEM: return "out of memory";
    case RC_ERR_CAPACITY: return "capacity exceeded (claims, table entries, events or batch size)";
    case RC_ERR_BUSY: return "an operation of this kind is still in flight";
    case RC_ERR_TOO_LARGE: return "size exceeds the fixed scratch of the no-allocation entry point (RC_NOALLOC_MAX_PAGES)";
    default: return "unknown error";
  }
}
extern "C" const char* rc_last_cuda_error(rc_ctx* c) { return c ? c->cuda_err.c_str() : ""; }


// ---- the entry point that allocates nothing (rc.h: rc_digest_blocks_noalloc) ---------------------------------------------
// The standalone checksum pass (k_move_hash_tma<DIGEST> + k_block_digest) needs scratch: the warp partial sums of every
// page, 128 B each.  rc_digest_blocks takes them from a context (cudaMalloc at rc_create); this variant takes them from
// a file-scope array, so that callers that may not allocate -- CUDA graph capture, serving loops, harnesses that forbid
// cudaMalloc -- have one entry point that needs no context and calls no allocating routine.  Every GPU that loads the
// library holds the 4 MiB until exit.  Every call shares the array; nothing in it has to start at zero (each partial the
// reduction reads is written by the same call's first kernel), and two calls that overlap on the GPU race on it.
static __device__ __align__(256) unsigned char g_noalloc_scratch[(size_t)RC_NOALLOC_MAX_PAGES * WPC * 2 * sizeof(u64)];

namespace {
struct NoAllocDev { bool ready = false; u64* scratch = nullptr; int sms = 0; };
constexpr int kNoAllocMaxDev = 64;
NoAllocDev g_noalloc_dev[kNoAllocMaxDev];
std::mutex g_noalloc_mu;
}  // namespace

extern "C" int rc_digest_blocks_noalloc(const void* src, uint32_t n_blocks, uint32_t layers, uint64_t page_bytes,
                                        uint64_t* d_out, uint64_t* e_out, void* stream) {
  if (n_blocks == 0) return RC_OK;
  if (!src || ((uintptr_t)src & 15) || !d_out || !e_out || !layers || !page_bytes || page_bytes % 4096 != 0 ||
      page_bytes > (1ull << 30) || layers > (1u << 20))
    return RC_ERR_INVALID;
  const u64 G = 2ull * layers, pages = (u64)n_blocks * G;
  if (pages > RC_NOALLOC_MAX_PAGES) return RC_ERR_TOO_LARGE;
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kNoAllocMaxDev) return RC_ERR_CUDA;
  NoAllocDev nd;
  {
    // set-up, once per device, with that device current: in host code the array's name is a host-side stand-in, not a
    // device address -- the kernels get the address cudaGetSymbolAddress returns for THIS device
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    NoAllocDev& slot = g_noalloc_dev[dev];
    if (!slot.ready) {
      void* p = nullptr;
      if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) return RC_ERR_CUDA;
      if (cudaDeviceGetAttribute(&slot.sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || slot.sms <= 0) return RC_ERR_CUDA;
      slot.scratch = (u64*)p;
      slot.ready = true;
    }
    nd = slot;
  }
  cudaStream_t s = (cudaStream_t)stream;
  const u32 grid = (u32)std::min<u64>(pages, 2ull * nd.sms);
  // 8 KiB (4 KiB for pages that are no multiple of 8 KiB) tiles x 4 stages: 32 / 16 KiB of dynamic shared memory, below the
  // 48 KiB that need no function attribute
  if (page_bytes % 8192 == 0)
    k_move_hash_tma<MV_DIGEST, 4, 8192, 1><<<grid, tma_threads<1>(), 4 * 8192, s>>>(
        nullptr, (u8*)src, nullptr, nd.scratch, n_blocks, (u32)G, 0, (u32)page_bytes, nullptr, nullptr, (u32)G, 1);
  else
    k_move_hash_tma<MV_DIGEST, 4, 4096, 1><<<grid, tma_threads<1>(), 4 * 4096, s>>>(
        nullptr, (u8*)src, nullptr, nd.scratch, n_blocks, (u32)G, 0, (u32)page_bytes, nullptr, nullptr, (u32)G, 1);
  if (cudaGetLastError() != cudaSuccess) return RC_ERR_CUDA;
  k_block_digest<<<warps_grid(n_blocks), 256, 0, s>>>(nd.scratch, nullptr, d_out, e_out, n_blocks, (u32)G, nullptr);
  if (cudaGetLastError() != cudaSuccess) return RC_ERR_CUDA;
  return RC_OK;
}
