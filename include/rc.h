/* rc.h -- C ABI of librc: claim-scoped offload and restoration of paged KV-cache
 * blocks on one B200 (sm_100a).
 *
 * What the path means is fixed by /root/reference/PAPER.md (P:Lnnn = line nnn):
 *   P:L25-27   running example and the accepted order  accept(C,P,>=448),
 *              materialized(C), offloaded(C), restore-required(C), same-claim
 *              load failure, restoration_failed(C),
 *              active_request_refused(blocking_claim_ids=[C]);
 *   P:L333     acceptance precedes every lifecycle event; refusal follows the
 *              same-claim restoration failure, before terminal handling;
 *   P:L337     failure injection is off by default, hits only CPU->GPU transfers,
 *              filters by claim id; unclaimed failures need a separate flag;
 *   P:L199     ambiguity fails closed: an error emits no claim outcome.
 * Byte layouts, checksum, allocator rule and code numbering are build-defined
 * (DESIGN.md "Readings").
 *
 * Conventions.  Every function returns 0 (RC_OK) or a negative call-level error;
 * nothing throws, nothing uses errno.  Batch calls also fill a caller-owned HOST
 * array int32_t status[n] (RC_ST_*).  Any status other than RC_ST_OK and
 * RC_ST_RESTORE_FAILED means: no event was emitted for that claim by that call and
 * its state is unchanged.  All pointer arguments are HOST pointers unless marked
 * DEVICE.  Calls without a _begin suffix are synchronous: on return the device work
 * is complete.  One caller thread per context.  A CUDA error poisons the context:
 * every later call returns RC_ERR_CUDA.  A call-level error (negative return) emits
 * no event and changes no claim (RC_ERR_CUDA excepted: the context is poisoned and claim state is then undefined).
 * There is no CPU fallback anywhere behind this
 * interface: every step of the path runs in the library's sm_100a kernels and its
 * copy-engine transfers.  Stream order: the library's streams are not ordered against
 * the caller's; writes the caller makes to pool_dev / fill_dev must have completed
 * (stream or device synchronise) before a call that reads them, and the library's
 * writes are complete when a synchronous call or rc_wait returns.
 * Environment: RC_CHECK=1 at rc_create turns on checked mode -- the work items of every gather / scatter launch are
 * validated on the device (pool block, work position, staged block in range) and rc_wait returns RC_ERR_CUDA if one was
 * not; RC_TRACE_LAUNCHES=1 prints per-launch device times on stderr; RC_TMA_VARIANT=<i> overrides the mover variant.
 */
#ifndef RC_H_
#define RC_H_
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct rc_ctx rc_ctx;

enum { RC_OK = 0, RC_ERR_INVALID = -1, RC_ERR_CUDA = -2, RC_ERR_NOMEM = -3, RC_ERR_CAPACITY = -4,
       RC_ERR_BUSY = -5, RC_ERR_TOO_LARGE = -6 /* rc_digest_blocks_noalloc: beyond its fixed scratch */ };

/* per-claim status */
enum { RC_ST_OK = 0, RC_ST_PRED_FALSE = 1, RC_ST_UNKNOWN_CLAIM = 2, RC_ST_BAD_STATE = 3,
       RC_ST_DUPLICATE_ID = 4, RC_ST_BAD_TABLE = 5, RC_ST_NO_FREE_BLOCKS = 6,
       RC_ST_NO_HOST_SPACE = 7, RC_ST_RESTORE_FAILED = 8, RC_ST_PROTECTED_CONFLICT = 9 };

/* event codes (the ordered claim-scoped outcome stream) */
enum { RC_EV_ACCEPTED = 1,          /* aux = N (predicate threshold), arg = P (prefix tokens)      */
       RC_EV_MATERIALIZED = 2,      /* aux = M (leading materialized tokens), arg = 0              */
       RC_EV_OFFLOADED = 3,         /* aux = nb (blocks offloaded), arg = chain checksum           */
       RC_EV_RESTORE_REQUIRED = 4,  /* aux = M (the lookup "hit"), arg = 0                 */
       RC_EV_LOAD_FAILED = 5,       /* aux = first bad block index, 0xFFFFFFFF = transfer error    */
       RC_EV_RESTORED = 6,          /* aux = nb, arg = chain checksum                              */
       RC_EV_RESTORATION_FAILED = 7,
       RC_EV_ACTIVE_REQUEST_REFUSED = 8, /* aux = 1 = |blocking_claim_ids|, arg = C; request form below */
       RC_EV_DEMOTED = 9, RC_EV_EXPIRED = 10, /* NEXT-3: the other claim-scoped outcomes of a failed restoration (arg = 0);
                                                 DEMOTED with arg = request id: a victim demoted by rc_make_room    */
       RC_EV_CONFLICT_REFUSED = 11 /* NEXT-3: active_request_refused(blocking_claim_ids) under hard protection:
                                      claim_id = a blocking claim, aux = RC_REFUSED_REQUEST | k, arg = request id */ };
/* request-level refusal (rc_restore_request): aux = RC_REFUSED_REQUEST | size of blocking_claim_ids, arg = request id */
#define RC_REFUSED_REQUEST 0x80000000u

/* claim states */
enum { RC_CS_ACCEPTED = 1, RC_CS_MATERIALIZED = 2, RC_CS_OFFLOADED = 3, RC_CS_RESIDENT_AGAIN = 4,
       RC_CS_REFUSED = 5, RC_CS_DEMOTED = 6, RC_CS_EXPIRED = 7 };
enum { RC_POLICY_REFUSE = 0, RC_POLICY_DEMOTE = 1, RC_POLICY_EXPIRE = 2 };

enum { RC_FAULT_XFER_ERROR = 1, RC_FAULT_BITFLIP = 2 };
enum { RC_FAULT_ALLOW_UNCLAIMED = 1 };

/* which data mover the gather / scatter launches use */
enum { RC_MOVER_AUTO = 0, RC_MOVER_LDG = 1 /* 16-byte register copies */, RC_MOVER_TMA = 2 /* bulk-copy smem ring */ };

typedef struct rc_event { uint64_t seq; uint64_t claim_id; uint32_t code; uint32_t aux; uint64_t arg; } rc_event;
typedef struct rc_fault { uint64_t claim_id; uint32_t kind; uint32_t param; } rc_fault;

typedef struct rc_config {
  uint32_t layers, kv_heads, head_dim, elem_bytes; /* elem_bytes: 1 (fp8) or 2 (bf16); bytes are never decoded */
  uint32_t block_size;                 /* tokens per block (BS), <= 255                               */
  uint32_t pool_blocks;                /* NB                                                          */
  uint32_t max_claims;                 /* live claims                                                 */
  uint32_t max_table_entries;          /* total block-table entries over all live claims              */
  uint32_t max_events;                 /* event ring capacity (records not yet drained)               */
  uint32_t staging_chunks;             /* ring depth per direction, >= 2                              */
  uint64_t staging_chunk_bytes;        /* rounded down to a multiple of blk = 2*L*page                */
  uint64_t host_store_bytes;           /* pinned host store, rounded down to a multiple of blk        */
  void*    pool_dev;   /* DEVICE, caller-owned: [layers][2][NB][BS][kv_heads][head_dim], 256-B aligned */
  uint8_t* fill_dev;   /* DEVICE, caller-owned u8[NB]: tokens materialized in each physical block     */
  /* cudaStream_t, caller-owned (e.g. torch); any may be NULL and is then created by the library.   */
  void*    stream_meta;     /* metadata kernels: their order on this stream is the order of calls    */
  void*    stream_gather;   /* offload: gather + digest kernels                                      */
  void*    stream_d2h;      /* offload: staging -> pinned host copies                                */
  void*    stream_scatter;  /* restore: scatter + digest kernels                                     */
  void*    stream_h2d;      /* restore: pinned host -> staging copies                                */
  uint32_t mover;           /* RC_MOVER_*                                                            */
  uint32_t grid_ctas;       /* CTAs of a gather / scatter launch; 0 = library default                */
  uint32_t dedup;           /* NEXT-2: 1 = content-addressed host store keyed by the 128-bit (d, e) digests: a block shared
                               between claims is held and crosses the link once       */
  uint32_t direct_offload;  /* NEXT-4 (experimental): 1 = the gather kernel stores straight into the mapped pinned
                               store (no staging, no copy engine); ignored with dedup                          */
  uint32_t tp_ranks, tp_rank; /* NEXT-4: TP-sharded KV: this context holds the kv_heads of rank
                               tp_rank of tp_ranks (<= 16); kv_heads above is the PER-RANK head count.  0 / 1 = off.
                               With tp_ranks > 1 OFFLOADED / RESTORED carry arg = 0 (chains are rank-local) so that
                               every rank emits the byte-identical stream; not combinable with dedup.          */
  uint32_t layer_major;     /* NEXT-4: 1 = layer-major streaming order.  A claim's host copy is laid out [g][block][page]
                               (g = layer*2 + kv: all its blocks' page 0, then page 1, ...) instead of [block][g][page], a
                               staging chunk is [g][item][page], and the copies of a chunk are issued plane by plane, so
                               layer 0 crosses the link first.  Digests, chains, statuses, allocation and events do not
                               change; rc_host_read returns the layer-major bytes; rc_host_store (a contiguous block) is
                               RC_ERR_INVALID; an injected BITFLIP's param indexes the host copy in its own layout.
                               Nothing is usable before the claim's verdict (RESTORED precedes use).  Not combinable
                               with dedup or direct_offload.                                                       */
} rc_config;

typedef struct rc_claim_info_t {
  uint64_t claim_id, chain, host_bytes;
  uint32_t state, P, N, M, nb, n_table;
} rc_claim_info_t;

typedef struct rc_stats {
  uint64_t bytes_d2h, bytes_h2d;         /* payload bytes moved over the host link                    */
  uint64_t claims_offloaded, claims_restored, claims_refused;
  uint64_t generic_failures;             /* unclaimed injected failures: a counter, never an outcome   */
  uint64_t host_used_bytes, free_blocks, events_emitted, kernel_launches;
  float    ms_gather, ms_scatter;        /* summed device time of the gather / scatter kernels         */
  float    ms_d2h, ms_h2d;               /* summed device time of the copies (copy-stream events)      */
  uint64_t gather_launches, scatter_launches, gather_blocks, scatter_blocks;
} rc_stats;

/* Creates a context.  page = BS*kv_heads*head_dim*elem_bytes must be a multiple of 4096
 * (checksum lanes).  The library owns: staging rings (device), pinned host store, claim
 * table, digests, allocator state, event ring, fault table.  All pool blocks start free. */
int rc_create(const rc_config* cfg, rc_ctx** out);
int rc_destroy(rc_ctx* ctx);

/* Allocator hand-over: blocks the caller already filled become "used" (ref 0), or go back
 * to free if no claim references them (claimed blocks are left alone). */
int rc_mark_used(rc_ctx* ctx, uint32_t n, const uint32_t* block_ids);
/* Convenience for callers that keep the materialization marks on the host: fill_dev[block_ids[i]] = values[i] (HOST
 * arrays; values <= block_size, ids < pool_blocks, else RC_ERR_INVALID and nothing is written).  The bytes cross PCIe in
 * the library's small-transfer path, not through a copy engine, so the call does not wait behind chunk copies in
 * flight.  Complete on return.  Writing fill_dev directly (it is caller-owned device memory) is equivalent. */
int rc_set_fill(rc_ctx* ctx, uint32_t n, const uint32_t* block_ids, const uint8_t* values);
int rc_mark_free(rc_ctx* ctx, uint32_t n, const uint32_t* block_ids);

/* a0. Records (C, P, N, block table) before any lifecycle event.  Table k is
 * bt_ids[bt_off[k] .. bt_off[k+1]) and must have ceil(P/BS) distinct in-range used blocks.
 * Emits ACCEPTED.  Statuses: OK, UNKNOWN_CLAIM (id 0 is reserved), DUPLICATE_ID, BAD_TABLE. */
int rc_accept(rc_ctx* ctx, uint32_t n, const uint64_t* claim_id, const uint32_t* prefix_tokens,
              const uint32_t* pred_min_tokens, const uint32_t* bt_off, const uint32_t* bt_ids,
              int32_t* status);

/* a1. Evaluates leading-prefix-at-least-N on the device from fill_dev: token t is materialized
 * iff (t mod BS) < fill[bt[t div BS]]; M = leading run; holds iff M >= N.
 * Emits MATERIALIZED for claims whose predicate holds; PRED_FALSE leaves the claim ACCEPTED. */
int rc_materialize(rc_ctx* ctx, uint32_t n, const uint64_t* claim_id, int32_t* status);

/* a1-a4. Gathers the nb = ceil(M/BS) leading blocks of every eligible claim (block-major, then
 * page g = layer*2 + kv) through the staging ring into the pinned host store, digests each
 * block while it streams, chains the digests per claim, drops the claim's references to ALL
 * its table blocks and emits OFFLOADED.  Host space is granted in batch order;
 * the first claim that does not fit and every later one get NO_HOST_SPACE. */
int rc_offload(rc_ctx* ctx, uint32_t n, const uint64_t* claim_id, int32_t* status);

/* a5-a8. For OFFLOADED claims: free blocks are granted in batch order against the free count
 * at entry (NO_FREE_BLOCKS for the first claim that does not fit and all later ones); served
 * claims take the lowest free ids ascending; host bytes are copied back, scattered into the
 * new blocks, re-digested and compared with the recorded digests and chain.  Emits, per claim
 * and consecutively, RESTORE_REQUIRED then RESTORED, or RESTORE_REQUIRED, LOAD_FAILED,
 * RESTORATION_FAILED, ACTIVE_REQUEST_REFUSED (status RESTORE_FAILED; the claim is terminal,
 * its new blocks are freed). */
int rc_restore(rc_ctx* ctx, uint32_t n, const uint64_t* claim_id, int32_t* status);

/* Split forms (BASELINE.json configs[4]: restore of batch k overlapped with the offload of the next batches on
 * separate streams).  _begin validates, enqueues the data movement and returns; rc_wait completes the operation: the
 * status array must stay valid until rc_wait fills it in.  which: 0 = offload, 1 = restore.
 * On return from a _begin, status[k] is final for the entries that were not served and -1 for the served ones; if no entry
 * is -1, nothing was opened and no rc_wait is owed for this call (rc_wait always completes the oldest operation that IS open).
 *   rc_offload_begin  enqueues a1-a3 and the chain on the gather / d2h streams.  Up to TWO offloads may be open; they
 *       run back to back, so the D2H direction stays busy while a slower restore is still in flight.  The claims stay
 *       referenced (their pool blocks are not free) until the offload is completed.  RC_ERR_BUSY with two open (one
 *       in dedup / direct_offload mode; in dedup mode the content store is looked up and extended by this call).
 *   rc_wait(ctx, 0)   completes the OLDEST open offload: waits for its transfer, then a4 -- reference drop, OFFLOADED.
 *   rc_restore_begin  a5 (grant, allocation of the new blocks, fault decision) takes place now; a6 and the scatter are
 *       enqueued on the h2d / scatter streams.  One restore may be in flight.  Blocks only until the plan is known.
 *   rc_wait(ctx, 1)   completes the restore: waits for its data movement, then a7-a8 -- verdicts, fill / release of
 *       the new blocks, RESTORE_REQUIRED and the outcome records; the host copy (its bytes in the pinned store) is
 *       given back here.
 * Between _begin and rc_wait the metadata stream is idle: accept / materialize / release of OTHER claims, rc_outcomes
 * and further _begin calls do not wait for the transfers.  Metadata steps execute in call order on one stream, so
 * every observable (statuses, allocation, events, seq numbers) equals the synchronous calls made in this order: an
 * offload at its rc_wait(0); a restore's plan at its _begin and its outcome at its rc_wait(1) (the oracle's
 * rco_restore_begin / rco_restore_end).  One decision of an offload is taken earlier than that: its host-space grant
 * (NO_HOST_SPACE) is evaluated at _begin, against the space held then -- never less strict than at its rc_wait(0).
 * The claims of an operation in flight answer BAD_STATE to every other call.
 * rc_test: *done = 1 if rc_wait(ctx, which) would not have to wait for data movement (the oldest open offload's gather
 * and D2H have finished / the restore's H2D and scatter have finished / nothing is in flight), else 0.  Never blocks. */
int rc_offload_begin(rc_ctx* ctx, uint32_t n, const uint64_t* claim_id, int32_t* status);
int rc_restore_begin(rc_ctx* ctx, uint32_t n, const uint64_t* claim_id, int32_t* status);
int rc_wait(rc_ctx* ctx, int which);
int rc_test(rc_ctx* ctx, int which, int* done);

/* NEXT-3.  rc_set_policy: what a failed restoration means for each named claim -- refusal
 * (default), demotion or expiry ("claim-scoped restoration failure/refusal, demotion, expiry");
 * a demoted / expired claim gets RESTORE_REQUIRED, LOAD_FAILED, RESTORATION_FAILED, DEMOTED | EXPIRED and is
 * terminal.  Unknown id or policy -> RC_ERR_INVALID, nothing changes.
 * rc_restore_request: the batch is ONE reuse request (request_id != 0) naming several claims.  Per-claim records
 * are as in rc_restore except that refusals are deferred: after all of them the request is refused once, by one
 * ACTIVE_REQUEST_REFUSED record per blocking claim in batch order (claim_id = the blocking claim,
 * aux = RC_REFUSED_REQUEST | k, arg = request_id) -- blocking_claim_ids is exactly the k claims whose restoration
 * failed under the refusal policy (smeared or partial attribution fails closed). */
int rc_set_policy(rc_ctx* ctx, uint32_t n, const uint64_t* claim_id, const uint32_t* policy);
int rc_restore_request(rc_ctx* ctx, uint64_t request_id, uint32_t n, const uint64_t* claim_id, int32_t* status);
int rc_restore_request_begin(rc_ctx* ctx, uint64_t request_id, uint32_t n, const uint64_t* claim_id, int32_t* status);

/* NEXT-4 (DESIGN.md 8 / R24): TP-sharded KV.  The pool is split by kv_head over tp_ranks ranks;
 * every rank makes the same calls with the same arguments on its shard (own digests, own chain, same block ids).  The
 * restoration verdict must be common, so a restore runs in two calls with the exchange in between:
 *   rc_tp_restore_verify  a5-a7 on this rank: plan, allocation, H2D, scatter, digests, LOCAL verdict.  Nothing is
 *       emitted and no block is released.  local[k] = { flags: RC_TP_SERVED | RC_TP_OK, bad }; status[k] is final for
 *       entries that were not served (as rc_restore) and -1 for served ones.  The records are also stored into every
 *       open peer mailbox (below).
 *   rc_tp_restore_commit  a8 on the merged verdict: ok = AND over ranks, bad = min over the failing ranks (k_tp_merge);
 *       fill / release of the new blocks, RESTORE_REQUIRED and the outcome records, statuses.  gathered = HOST
 *       [ranks][n] records of all ranks in rank order (e.g. one all-gather), or NULL to read this rank's mailbox: then
 *       every rank must have completed its verify (one barrier); RC_ERR_BUSY if a peer has not published yet -- the
 *       library never waits inside a kernel for another rank.  RC_ERR_INVALID if the ranks disagree on which entries
 *       were served (they did not make the same call); nothing is applied then and the commit may be repeated.
 * Between the two calls rc_wait(1), rc_restore*, rc_make_room return RC_ERR_BUSY / RC_ERR_INVALID.
 * Mailboxes (NVLink / NVSwitch path): rc_tp_mailbox returns this rank's mailbox (DEVICE); a peer rank is attached with
 * rc_tp_set_peer (a device pointer valid in this process) or rc_tp_ipc_handle / rc_tp_open_peer (64-byte CUDA IPC
 * handle, for one process per GPU). */
enum { RC_TP_SERVED = 1, RC_TP_OK = 2 };
typedef struct rc_tp_verdict { uint32_t flags, bad; } rc_tp_verdict;
int rc_tp_restore_verify(rc_ctx* ctx, uint32_t n, const uint64_t* claim_id, int32_t* status, rc_tp_verdict* local);
int rc_tp_restore_commit(rc_ctx* ctx, uint32_t n, uint32_t ranks, const rc_tp_verdict* gathered, int32_t* status);
int rc_tp_mailbox(rc_ctx* ctx, void** mailbox_dev, uint64_t* bytes);
int rc_tp_set_peer(rc_ctx* ctx, uint32_t rank, void* mailbox_dev /* DEVICE */);
int rc_tp_ipc_handle(rc_ctx* ctx, void* handle64 /* HOST, 64 bytes out */);
int rc_tp_open_peer(rc_ctx* ctx, uint32_t rank, const void* handle64 /* HOST, 64 bytes */);

/* NEXT-3, allocator-side protection (P:L85 victim_exclusion_before_violation, explicit_conflict_action,
 * blocking_claim_ids, claim_demoted_before_loss; P:L103 hard_protected; P:L270 allocator_hook).
 * rc_protect: marks live (non-terminal) claims hard_protected (on = 1) or not (0).  The protected resident footprint is
 * the union of the block tables of protected claims (rc_protected_map copies it out as u8[NB]); it follows a claim
 * through offload and restore.  Unknown / terminal id or on > 1 -> RC_ERR_INVALID, nothing changes.
 * rc_make_room: an active request (request_id != 0) needs `need_blocks` free blocks.  If they are free already:
 * status OK, nothing happens.  Otherwise the victim candidates are the live claims that hold a table, unprotected
 * first, then protected, each group in acceptance order; evicting a claim frees the blocks whose last holder it is.
 * If a prefix of the UNPROTECTED candidates suffices, exactly that prefix is demoted: DEMOTED(C, aux = table blocks
 * released, arg = request_id) is emitted before the claim's references are dropped; the claims become terminal;
 * status OK, ids = the demoted claims.  If the need could only be met from a protected footprint, nothing is evicted
 * and no block changes hands: status RC_ST_PROTECTED_CONFLICT, ids = blocking_claim_ids = the protected claims the
 * walk had to enter, one RC_EV_CONFLICT_REFUSED record each.  No protected claim in the way: RC_ST_NO_FREE_BLOCKS, no
 * event.  n_ids receives the number of ids (may exceed cap).  RC_ERR_BUSY while an offload or restore is in flight. */
int rc_protect(rc_ctx* ctx, uint32_t n, const uint64_t* claim_id, const uint32_t* on);
int rc_make_room(rc_ctx* ctx, uint64_t request_id, uint32_t need_blocks, int32_t* status, uint64_t* ids, uint32_t cap,
                 uint32_t* n_ids);
int rc_protected_map(rc_ctx* ctx, uint8_t* prot /* HOST u8[NB] */);

/* Drains up to cap not-yet-returned events of completed calls, in seq order. */
int rc_outcomes(rc_ctx* ctx, rc_event* buf, uint64_t cap, uint64_t* n_out);

/* Replaces the armed fault set (n = 0 disarms; default is disarmed).  A fault fires only in
 * rc_restore (CPU->GPU) and only for the claim it names, once.  Entries with claim_id 0 are
 * rejected (RC_ERR_INVALID) unless flags has RC_FAULT_ALLOW_UNCLAIMED; they only bump
 * rc_stats.generic_failures. */
int rc_set_faults(rc_ctx* ctx, uint32_t n, const rc_fault* faults, uint32_t flags);

/* Forgets claims in any state, dropping block references and host bytes.  Emits nothing. */
int rc_release(rc_ctx* ctx, uint32_t n, const uint64_t* claim_id, int32_t* status);

/* Introspection (tests, parity). */
int rc_claim_info(rc_ctx* ctx, uint64_t claim_id, rc_claim_info_t* out);
int rc_claim_blocks(rc_ctx* ctx, uint64_t claim_id, uint32_t* ids, uint32_t cap, uint32_t* n);
/* d: the recorded per-block checksums (chained into `chain`); e (may be NULL): the second digests -- (d[i], e[i]) is
 * the 128-bit content key of block i (DESIGN.md "Checksum" R22). */
int rc_claim_digests(rc_ctx* ctx, uint64_t claim_id, uint64_t* d, uint64_t* e, uint32_t cap, uint32_t* n);
/* Copies the claim's host bytes (its own layout) to dst if cap suffices; *bytes = their size (0: none held).  RC_ERR_BUSY while
 * the claim's offload is in flight. */
int rc_host_read(rc_ctx* ctx, uint64_t claim_id, void* dst, uint64_t cap, uint64_t* bytes);
/* Borrowed, READ-ONLY view of the claim's host copy: *p = the pinned-store address of the claim's block `block` (offload
 * order: block-major, then page g = layer*2 + kv), *contiguous_bytes = how many bytes from there belong to the claim and
 * are contiguous (a claim's bytes may be split over several extents of the store).  Valid until the claim is restored,
 * released or offloaded again; RC_ERR_BUSY while the claim's offload is in flight; RC_ERR_INVALID if the claim holds no
 * such host block.  (rc_host_read is the copying form.) */
int rc_host_store(rc_ctx* ctx, uint64_t claim_id, uint32_t block, const void** p, uint64_t* contiguous_bytes);
/* Completes every in-flight operation (every open offload in _begin order as rc_wait(0), then rc_wait(1)) and drains
 * the library's streams.  rc_offload (synchronous) likewise completes the offloads opened before it, then its own. */
int rc_sync(rc_ctx* ctx);
int rc_pool_state(rc_ctx* ctx, uint8_t* used /*NB*/, uint32_t* ref /*NB*/);
int rc_stats_get(rc_ctx* ctx, rc_stats* out);
int rc_stats_reset(rc_ctx* ctx);

/* Host-link ceiling: best-of-`reps` cudaMemcpyAsync of `bytes` between the context's pinned
 * store and its staging ring; direction 0 = D2H, 1 = H2D, 2 = both at once (sum).  GB/s.  The copies write over the
 * pinned store and the staging ring, so the call is refused with RC_ERR_BUSY while an operation is in flight or
 * any claim holds host bytes. */
int rc_measure_link(rc_ctx* ctx, uint64_t bytes, int direction, int reps, double* gbs);

/* Standalone checksum of `n_blocks` contiguous blocks at DEVICE address src (offload order):
 * the read-only digest pass used to report the checksum against the HBM roofline.  digests / digests2
 * are HOST arrays (d and e of each block; either may be NULL); ms (may be NULL) receives the device
 * time of the digest kernel. */
int rc_digest_blocks(rc_ctx* ctx, const void* src_dev, uint32_t n_blocks, uint64_t* digests, uint64_t* digests2, float* ms);

/* The one entry point that ALLOCATES NOTHING -- for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  Same result as rc_digest_blocks (d and e of `n_blocks` contiguous
 * blocks at DEVICE address src_dev, offload order: block-major, then page g = layer*2 + kv), but: no context; geometry
 * passed in (blk = 2*layers*page_bytes, page_bytes % 4096 == 0, src_dev 16-byte aligned); d_out_dev / e_out_dev are
 * caller-owned DEVICE arrays of n_blocks u64; the two kernels are enqueued on `stream` (a cudaStream_t, NULL = the default
 * stream) and the call returns without synchronising -- the outputs are complete in stream order.  The scratch the pass
 * needs (128 B of partial sums per page) lives in a fixed 4 MiB device array inside the library, which every GPU that
 * loads the library holds until exit: n_blocks * 2 * layers <= RC_NOALLOC_MAX_PAGES, beyond that RC_ERR_TOO_LARGE and
 * nothing is enqueued (split the range, or use rc_digest_blocks).  Calls no cudaMalloc / cudaFree / allocating routine;
 * the first call on a device looks up the array's address on that device (the device must be current, as for every
 * call).  Every call on a device shares the array: nothing in it has to start at zero, but calls that may overlap on
 * the GPU (different streams, no ordering between them) race on it -- order them on one stream or by events. */
#define RC_NOALLOC_MAX_PAGES 32768u
int rc_digest_blocks_noalloc(const void* src_dev, uint32_t n_blocks, uint32_t layers, uint64_t page_bytes,
                             uint64_t* d_out_dev, uint64_t* e_out_dev, void* stream);

/* NEXT-1: the paper's artifact analyzer as a device pass.  Validates an event
 * array (HOST, n records in stream order; may contain the harness marker codes RC_EV_USE and
 * RC_EV_REQUEST_FINISHED) against the per-claim language
 *   ACCEPTED MATERIALIZED ( OFFLOADED RESTORE_REQUIRED ( RESTORED USE* | LOAD_FAILED RESTORATION_FAILED
 *                                                          ( REFUSED | DEMOTED | EXPIRED ) ) )*
 * (any prefix valid; only REQUEST_FINISHED may follow REFUSED; REQUEST_FINISHED also ends ACCEPTED /
 * MATERIALIZED / RESTORED), seq strictly increasing, no event with claim id 0, REFUSED carrying [C] (aux 1, arg C)
 * or belonging to a request run (aux = RC_REFUSED_REQUEST | k, arg = request id: k consecutive records that name
 * exactly the k claims whose restoration failed and is unanswered).
 * report->ok = 1 iff the whole stream is accepted; first_bad_index = stream position of the first
 * violation (UINT64_MAX if none).  claims (HOST, may be NULL) receives up to cap per-claim records in
 * unspecified order: final automaton state, gate bits (RC_GATE_FAILURE: the claim's subsequence ends with
 * the seven steps of P:L27; RC_GATE_OBSERVATION: path A; both 0 unless the stream is valid),
 * its first violating position.  NEXT-3 adds: DEMOTED with arg = request id from ACCEPTED / MATERIALIZED / RESTORED (a
 * victim of rc_make_room; DEMOTED after RESTORATION_FAILED keeps arg 0), and RC_EV_CONFLICT_REFUSED (aux =
 * RC_REFUSED_REQUEST | k, arg = request id) as a self-loop of a resident claim, k consecutive records naming k
 * different claims.  n <= 2^30 events (RC_ERR_INVALID above).  Needs no context; allocates and frees its own
 * device memory. */
enum { RC_EV_USE = 100, RC_EV_REQUEST_FINISHED = 101 };
enum { RC_GATE_FAILURE = 1, RC_GATE_OBSERVATION = 2 };
typedef struct rc_trace_claim { uint64_t claim_id; uint64_t first_bad; uint32_t state; uint32_t gates; uint32_t n_events; uint32_t pad; } rc_trace_claim;
typedef struct rc_trace_report {
  uint64_t first_bad_index, n_events, n_claims, n_failure_gate, n_observation_gate;
  uint32_t ok, pad;
  float ms_kernels;       /* device time of the four validator kernels */
  float ms_total;         /* including the H2D of the events and the D2H of the records */
} rc_trace_report;
int rc_validate_trace(const rc_event* events, uint64_t n, rc_trace_report* report, rc_trace_claim* claims, uint64_t cap);

const char* rc_strerror(int err);
const char* rc_last_cuda_error(rc_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif
