// rc_oracle.cpp -- ORACLE (test infrastructure, not the product).
//
// Plain single-threaded C++17 statement of what the claim-scoped KV offload /
// restore path computes.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load this library.  It shares no
// source, header, table or helper with paper_2606_01387_b200/csrc (constants
// are restated here on purpose).
//
// Passages followed (P:Lnnn = /root/reference/PAPER.md line nnn):
//   P:L25-27   running example: accept(C,P,leading-prefix-at-least-448),
//              materialized(C), offloaded(C), restore-required(C), same-claim
//              load failure, restoration_failed(C),
//              active_request_refused(blocking_claim_ids=[C]).
//   P:L333     "accepted" precedes lifecycle events; "refused" is emitted after
//              the same-claim restoration failure and before terminal handling.
//   P:L337     failure injection: off by default, CPU->GPU only, claim-id
//              filter, unclaimed failures need a separate flag.
//   P:L358-380 witness paths A (success) and B (same-claim failure).
//   P:L384     path C: only the target claim is attributed.
//   P:L199     ambiguity fails closed: an error status emits no event.
// Everything the paper leaves open (byte layout, checksum, allocator, codes) is
// build-defined: DESIGN.md "Readings" R1..R28.  Pins: tests/test_oracle_*.py.
// Parity unpinned (beyond GPU==oracle): status- and event-code numbering, aux/arg
// payload choice, one-shot fault consumption (R18), the NO_FREE_BLOCKS /
// NO_HOST_SPACE refusal policy (R7, R26), the victim order inside a group (R23).
#include <cstdint>
#include <cstring>
#include <cstdlib>
#include <vector>
#include <map>
#include <set>
#include <algorithm>

typedef uint64_t u64;
typedef uint32_t u32;
typedef uint8_t u8;

// ---- checksum (build-defined, reading R22) ---------------
// All arithmetic mod 2^64 (products: the full 128 bits), memory read as little-endian u64.
static const u64 K1 = 0x9E3779B97F4A7C15ull;  // floor(2^64/phi)
static const u64 K2 = 0x6A09E667F3BCC909ull;  // frac(sqrt 2) | 1
static const u64 KA = 0xBB67AE8584CAA73Bull;  // frac(sqrt 3), odd
static const u64 K3 = 0x3C6EF372FE94F82Bull;  // frac(sqrt 5)
static const u64 K4 = 0xA54FF53A5F1D36F1ull;  // frac(sqrt 7)
static const u64 K5 = 0x510E527FADE682D1ull;  // frac(sqrt 11)

static u64 mixL(u64 x) { u64 y = x ^ (x >> 32); y *= K2; return y ^ (y >> 29); }
static u64 mixF(u64 x) { u64 y = mixL(x); y *= K1; return y ^ (y >> 32); }
// mum(x, y): the 128-bit product x*y folded to 64 bits, low half XOR high half.  Unlike a
// multiplication by an odd constant mod 2^64 it carries a difference in ANY input bit into
// low and high output bits alike, and by an amount that depends on the other factor.
static u64 mum(u64 x, u64 y) {
  unsigned __int128 p = (unsigned __int128)x * y;
  return (u64)p ^ (u64)(p >> 64);
}

static u64 load64le(const u8* p) {
  u64 v = 0;
  for (int i = 7; i >= 0; --i) v = (v << 8) | p[i];
  return v;
}

// One page = V = page_bytes/16 vectors (a, b) of two little-endian u64 words.
// 256 lanes; lane t folds vectors t, t+256, t+512, ... in increasing order, in two
// independent families: h (the checksum) and g (the content-key extension).
struct Dig2 { u64 d, e; };
static Dig2 page_digest2(const u8* pg, u64 page_bytes) {
  u64 V = page_bytes / 16;
  Dig2 out = {0, 0};
  for (u64 lane = 0; lane < 256; ++lane) {
    u64 h = (lane + 1) * K1, g = (lane + 1) * K4;
    for (u64 v = lane; v < V; v += 256) {
      u64 a = load64le(pg + 16 * v), b = load64le(pg + 16 * v + 8);
      h = mum(a ^ K2, b ^ h);
      g = mum(b ^ K5, a ^ g);
    }
    out.d += mixL(h);
    out.e += mixL(g);
  }
  return out;
}

// A block in offload order: 2L pages, page g = l*2 + kv.  d = the 64-bit per-block checksum that is
// chained and verified (BASELINE.json north_star (d)); e = a second, independent 64-bit digest of the
// same bytes: (d, e) is the 128-bit content key of the dedup store, and verify compares it too.
static Dig2 block_digest2(const u8* blk, u32 n_pages, u64 page_bytes) {
  u64 s = 0, t = 0;
  for (u32 g = 0; g < n_pages; ++g) {
    Dig2 p = page_digest2(blk + (u64)g * page_bytes, page_bytes);
    s += mixL(p.d ^ ((u64)(g + 1) * K3));
    t += mixL(p.e ^ ((u64)(g + 1) * K5));
  }
  Dig2 out = {mixF(s), mixF(t)};
  return out;
}

static u64 chain_seed(u64 claim_id) { return mixF(claim_id ^ K3); }
static u64 chain_of(u64 claim_id, const u64* d, u32 nb) {
  u64 h = chain_seed(claim_id);
  for (u32 i = 0; i < nb; ++i) h = h * KA + d[i];
  return h;
}

// ---- codes (restated; the ABI header of the product is not included) --------
enum { EV_ACCEPTED = 1, EV_MATERIALIZED = 2, EV_OFFLOADED = 3, EV_RESTORE_REQUIRED = 4,
       EV_LOAD_FAILED = 5, EV_RESTORED = 6, EV_RESTORATION_FAILED = 7,
       EV_ACTIVE_REQUEST_REFUSED = 8,
       EV_DEMOTED = 9, EV_EXPIRED = 10,     // NEXT-3: the other claim-scoped outcomes of a failed restoration (Table "offloadable")
       EV_CONFLICT_REFUSED = 11 };          // NEXT-3: active_request_refused(blocking_claim_ids) under hard protection
enum { POL_REFUSE = 0, POL_DEMOTE = 1, POL_EXPIRE = 2 };
static const u32 REQ_FLAG = 0x80000000u;     // REFUSED.aux of a request-level refusal: flag | size of blocking_claim_ids
enum { ST_OK = 0, ST_PRED_FALSE = 1, ST_UNKNOWN_CLAIM = 2, ST_BAD_STATE = 3, ST_DUPLICATE_ID = 4,
       ST_BAD_TABLE = 5, ST_NO_FREE_BLOCKS = 6, ST_NO_HOST_SPACE = 7, ST_RESTORE_FAILED = 8,
       ST_PROTECTED_CONFLICT = 9 };
enum { CS_ACCEPTED = 1, CS_MATERIALIZED = 2, CS_OFFLOADED = 3, CS_RESIDENT_AGAIN = 4, CS_REFUSED = 5,
       CS_DEMOTED = 6, CS_EXPIRED = 7 };
enum { FK_XFER_ERROR = 1, FK_BITFLIP = 2 };
enum { FF_ALLOW_UNCLAIMED = 1 };
enum { E_OK = 0, E_INVALID = -1 };

struct Event { u64 seq, claim_id; u32 code, aux; u64 arg; };   // 32 bytes
struct Fault { u64 claim_id; u32 kind, param; };
struct ClaimInfo { u64 claim_id, chain, host_bytes; u32 state, P, N, M, nb, n_table; };

typedef std::pair<u64, u64> Key;   // 128-bit content key (d, e) of one block

struct Claim {
  u32 state = 0, P = 0, N = 0, M = 0, nb = 0, policy = 0;
  u32 protect = 0;            // NEXT-3: hard_protected -- its table is never a victim
  u64 order = 0;              // acceptance sequence number: the victim order
  std::vector<u32> bt;        // current block table
  std::vector<u64> d;         // per-block checksums recorded at offload (chained)
  std::vector<u64> e;         // per-block second digests recorded at offload ((d, e) = content key)
  u64 chain = 0;
  std::vector<u8> host;       // claim-scoped host copy (nb*blk bytes)
  std::vector<Key> hkeys;     // dedup mode (NEXT-2): the claim's blocks as keys into the content-addressed store
  bool in_flight = false;     // split form: between rco_restore_begin and rco_restore_end the claim answers BAD_STATE (rc.h)
};

struct Verdict { u32 flags, bad; };                     // flags: 1 = served, 2 = locally ok; bad = first bad block / 0xFFFFFFFF
enum { V_SERVED = 1, V_OK = 2 };

struct Ctx {
  u32 L, H, D, e, BS, NB;
  u64 page, blk, host_cap, host_used = 0;
  u8* pool;                   // caller-owned host mirror [L][2][NB][page]
  u8* fill;                   // caller-owned u8[NB]
  std::vector<u8> used;
  std::vector<u32> ref;
  std::map<u64, Claim> claims;
  std::vector<Fault> faults; u32 fault_flags = 0;
  std::vector<Event> events; u64 drained = 0;
  u64 generic_failures = 0;
  u64 accept_seq = 0;
  // NEXT-4: TP mode and the restore that waits between its two phases for the merged verdict
  u32 tp_ranks = 0;
  bool tp_pending = false; std::vector<u64> tp_ids; std::vector<void*> tp_served;
  std::vector<Verdict> split_v; u64 split_request = 0;     // split form of restore: phase-1 verdicts and the request id
  // NEXT-2: content-addressed host store keyed by block digest, so blocks shared between claims
  // are held (and cross the link) once.  DESIGN.md "Dedup".
  bool dedup = false;
  bool layer_major = false;                             // NEXT-4: host copy laid out [g][block][page] (DESIGN R28)
  std::map<Key, std::pair<std::vector<u8>, u32>> store;   // (d, e) -> (blk bytes, references)
  u64 link_d2h = 0, link_h2d = 0;                          // bytes that have to cross the host link, by definition
  void emit(u64 c, u32 code, u32 aux, u64 arg) {
    Event ev; ev.seq = events.size(); ev.claim_id = c; ev.code = code; ev.aux = aux; ev.arg = arg;
    events.push_back(ev);
  }
  u8* page_ptr(u32 g, u32 b) { return pool + ((u64)g * NB + b) * page; }
};

static u32 ceil_div(u32 a, u32 b) { return (a + b - 1) / b; }

// accept(C,P,N,bt): "first accepted by a mechanism that records C, P, and
// the predicate"; P:L199 duplicate ownership / ambiguity -> no claim outcome.
static int do_accept(Ctx* c, u64 id, u32 P, u32 N, const u32* bt, u32 nbt) {
  if (id == 0) return ST_UNKNOWN_CLAIM;                 // 0 is reserved: "no claim"
  if (c->claims.count(id)) return ST_DUPLICATE_ID;
  if (P == 0 || N == 0 || N > P) return ST_BAD_TABLE;
  if (nbt != ceil_div(P, c->BS)) return ST_BAD_TABLE;
  for (u32 i = 0; i < nbt; ++i) {
    if (bt[i] >= c->NB || !c->used[bt[i]]) return ST_BAD_TABLE;
    for (u32 j = 0; j < i; ++j) if (bt[j] == bt[i]) return ST_BAD_TABLE;
  }
  Claim cl; cl.state = CS_ACCEPTED; cl.P = P; cl.N = N; cl.bt.assign(bt, bt + nbt); cl.order = c->accept_seq++;
  for (u32 i = 0; i < nbt; ++i) c->ref[bt[i]]++;
  c->claims[id] = cl;
  c->emit(id, EV_ACCEPTED, N, P);
  return ST_OK;
}

// Predicate by its token-level definition (DESIGN R2): token t of the prefix is
// materialized iff (t mod BS) < fill[bt[t div BS]];  M = length of the leading
// run of materialized tokens;  leading-prefix-at-least-N holds iff M >= N
// (">=" because hit=448 with predicate 448 is served).
static u32 leading_materialized(Ctx* c, const Claim& cl) {
  u32 m = 0;
  while (m < cl.P && (m % c->BS) < c->fill[cl.bt[m / c->BS]]) ++m;
  return m;
}

static int do_materialize(Ctx* c, u64 id) {
  auto it = c->claims.find(id);
  if (it == c->claims.end()) return ST_UNKNOWN_CLAIM;   // post-hoc naming rejected
  Claim& cl = it->second;
  if (cl.state != CS_ACCEPTED) return ST_BAD_STATE;
  u32 M = leading_materialized(c, cl);
  if (M < cl.N) return ST_PRED_FALSE;                   // no event
  cl.M = M; cl.nb = ceil_div(M, c->BS); cl.state = CS_MATERIALIZED;
  c->emit(id, EV_MATERIALIZED, M, 0);
  return ST_OK;
}

static void drop_refs(Ctx* c, Claim& cl) {
  for (u32 b : cl.bt) { if (c->ref[b] > 0 && --c->ref[b] == 0) c->used[b] = 0; }
  cl.bt.clear();
}

static std::vector<u8> host_bytes_of(Ctx* c, const Claim& cl) {     // the claim-logical host copy
  if (!c->dedup) return cl.host;
  std::vector<u8> out;
  for (const Key& k : cl.hkeys) { const auto& b = c->store[k].first; out.insert(out.end(), b.begin(), b.end()); }
  return out;
}
static u64 host_size_of(Ctx* c, const Claim& cl) { return c->dedup ? (u64)cl.hkeys.size() * c->blk : (u64)cl.host.size(); }
static void drop_host(Ctx* c, Claim& cl) {
  if (c->dedup) {
    for (const Key& k : cl.hkeys) { auto it = c->store.find(k); if (--it->second.second == 0) { c->store.erase(it); c->host_used -= c->blk; } }
    cl.hkeys.clear();
  } else {
    c->host_used -= cl.host.size();
    std::vector<u8>().swap(cl.host);
  }
}

// Where page g of the claim's block i sits in its host copy (nb blocks).  Block-major (default): blocks one after the
// other, each its 2L pages.  Layer-major (NEXT-4, DESIGN R28): all blocks' page 0, then all blocks' page 1, ...
static u64 host_page_offset(const Ctx* c, u32 nb, u32 i, u32 g) {
  return c->layer_major ? ((u64)g * nb + i) * c->page : (u64)i * c->blk + (u64)g * c->page;
}
// block i of a host copy as contiguous bytes, pages g = 0 .. 2L-1
static std::vector<u8> block_of(const Ctx* c, const std::vector<u8>& host, u32 nb, u32 i) {
  std::vector<u8> out(c->blk);
  for (u32 g = 0; g < 2 * c->L; ++g) memcpy(out.data() + (u64)g * c->page, host.data() + host_page_offset(c, nb, i, g), c->page);
  return out;
}

// offload: P:L343-346 (E2-E5).  Host bytes = concatenation, block-major,
// then page g = l*2+kv (layer-major mode: see above).  Never failed by injection (CPU->GPU only).
static void do_offload_one(Ctx* c, u64 id, Claim& cl) {
  u32 G = 2 * c->L;
  cl.host.resize((u64)cl.nb * c->blk);
  for (u32 i = 0; i < cl.nb; ++i)
    for (u32 g = 0; g < G; ++g)
      memcpy(cl.host.data() + host_page_offset(c, cl.nb, i, g), c->page_ptr(g, cl.bt[i]), c->page);
  cl.d.resize(cl.nb); cl.e.resize(cl.nb);
  for (u32 i = 0; i < cl.nb; ++i) {
    std::vector<u8> blk = block_of(c, cl.host, cl.nb, i);   // the block's 2L pages, g ascending: what the digest is defined on
    Dig2 x = block_digest2(blk.data(), G, c->page);
    cl.d[i] = x.d; cl.e[i] = x.e;
  }
  cl.chain = chain_of(id, cl.d.data(), cl.nb);
  if (c->dedup) {                                         // keep one copy per distinct block content
    cl.hkeys.clear();
    for (u32 i = 0; i < cl.nb; ++i) {
      const Key key(cl.d[i], cl.e[i]);
      cl.hkeys.push_back(key);
      auto it = c->store.find(key);
      if (it != c->store.end()) { it->second.second++; continue; }
      const u8* b = cl.host.data() + (u64)i * c->blk;
      c->store[key] = std::make_pair(std::vector<u8>(b, b + c->blk), 1u);
      c->host_used += c->blk; c->link_d2h += c->blk;
    }
    std::vector<u8>().swap(cl.host);
  } else {
    c->host_used += cl.host.size(); c->link_d2h += cl.host.size();
  }
  drop_refs(c, cl);
  cl.state = CS_OFFLOADED;
  c->emit(id, EV_OFFLOADED, cl.nb, c->tp_ranks > 1 ? 0 : cl.chain);
}

static void do_offload(Ctx* c, u32 n, const u64* ids, int32_t* st) {
  bool full = false;                                    // prefix rule (DESIGN R7)
  u64 worst = c->host_used;                             // space is granted as if every block were new (dedup charges less)
  for (u32 k = 0; k < n; ++k) {
    auto it = c->claims.find(ids[k]);
    if (it == c->claims.end()) { st[k] = ST_UNKNOWN_CLAIM; continue; }
    Claim& cl = it->second;
    if (cl.state != CS_MATERIALIZED && cl.state != CS_RESIDENT_AGAIN) { st[k] = ST_BAD_STATE; continue; }
    if (full || worst + (u64)cl.nb * c->blk > c->host_cap) { full = true; st[k] = ST_NO_HOST_SPACE; continue; }
    worst += (u64)cl.nb * c->blk;
    do_offload_one(c, ids[k], cl);
    st[k] = ST_OK;
  }
}

// restore: P:L347-351 (E6-E9) on success; P:L353-356, P:L376-380 on same-claim
// failure.  The call works in the phases DESIGN R6/R7 fix:
//   1. eligibility in batch order (state must be OFFLOADED: restore-after-use and
//      double restore are BAD_STATE);
//   2. free-block prefix rule against the free count at call entry;
//   3. every served claim, in batch order, takes the next nb lowest free ids;
//   4. per served claim, batch order: RESTORE_REQUIRED, fault decision (first armed
//      entry whose id == C, one-shot; other ids have no effect: P:L25, P:L463,
//      P:L493), write + re-digest + compare, verdict events;
//   5. blocks of failed claims are freed after step 4 of that claim.
// request_id == 0: every claim is its own reuse request (blocking_claim_ids=[C]).  request_id != 0 (NEXT-3): the
// batch is ONE reuse request naming several claims; its refusal is emitted once, after the per-claim records, as
// one REFUSED record per failed claim (claim_id = the blocking claim, aux = REQ_FLAG | size of the failed subset,
// arg = request id) -- blocking_claim_ids is exactly the failed subset ("smeared" ids fail closed).
// The call is written in two phases so that a TP-sharded deployment (NEXT-4; below) can put the
// cross-rank verdict merge between them; rco_restore runs them back to back with the local verdicts.

// phase 1: steps 1-3 and, of step 4, everything but the events: fault decision, write, re-digest, LOCAL verdict
static void restore_verify(Ctx* c, u32 n, const u64* ids, int32_t* st, std::vector<Claim*>& served, std::vector<Verdict>& v) {
  u32 G = 2 * c->L;
  served.assign(n, nullptr);
  v.assign(n, Verdict{0, 0xFFFFFFFFu});
  u64 nfree = 0;
  for (u32 b = 0; b < c->NB; ++b) nfree += !c->used[b];
  u64 need = 0; bool full = false;
  for (u32 k = 0; k < n; ++k) {
    auto it = c->claims.find(ids[k]);
    if (it == c->claims.end()) { st[k] = ST_UNKNOWN_CLAIM; continue; }
    Claim& cl = it->second;
    bool dup = false;
    for (u32 j = 0; j < k; ++j) if (served[j] == &cl) dup = true;
    if (cl.state != CS_OFFLOADED || dup || cl.in_flight) { st[k] = ST_BAD_STATE; continue; }
    if (full || need + cl.nb > nfree) { full = true; st[k] = ST_NO_FREE_BLOCKS; continue; }
    need += cl.nb; served[k] = &cl; st[k] = ST_OK;
  }
  u32 cursor = 0;                                       // step 3: lowest free ids, ascending
  for (u32 k = 0; k < n; ++k) {
    if (!served[k]) continue;
    Claim& cl = *served[k];
    cl.bt.clear();
    while (cl.bt.size() < cl.nb) {
      while (c->used[cursor]) ++cursor;
      c->used[cursor] = 1; c->ref[cursor] = 1; cl.bt.push_back(cursor);
    }
  }
  std::set<Key> call_keys;
  for (u32 k = 0; k < n; ++k) {
    if (!served[k]) continue;
    Claim& cl = *served[k]; u64 id = ids[k];
    int fi = -1;
    for (size_t f = 0; f < c->faults.size(); ++f) if (c->faults[f].claim_id == id) { fi = (int)f; break; }
    Fault flt{0, 0, 0};
    if (fi >= 0) { flt = c->faults[fi]; c->faults.erase(c->faults.begin() + fi); }
    bool ok; u32 bad = 0xFFFFFFFFu;
    if (flt.kind == FK_XFER_ERROR) {
      ok = false;                                       // nothing is written to the pool
    } else {
      std::vector<u8> staged = host_bytes_of(c, cl);    // host copy itself stays intact
      if (c->dedup && flt.kind != FK_BITFLIP) {           // one transfer per distinct block of the call; a corrupted
        for (const Key& kk : cl.hkeys) if (call_keys.insert(kk).second) c->link_h2d += c->blk;   // copy is private to its claim
      } else c->link_h2d += staged.size();
      if (flt.kind == FK_BITFLIP && !staged.empty()) staged[flt.param % staged.size()] ^= 0x01;
      std::vector<u64> d2(cl.nb), e2(cl.nb);
      for (u32 i = 0; i < cl.nb; ++i) {
        for (u32 g = 0; g < G; ++g)
          memcpy(c->page_ptr(g, cl.bt[i]), staged.data() + host_page_offset(c, cl.nb, i, g), c->page);
        u32 rem = cl.M - i * c->BS;
        c->fill[cl.bt[i]] = (u8)(rem < c->BS ? rem : c->BS);
        std::vector<u8> blk = block_of(c, staged, cl.nb, i);
        Dig2 x = block_digest2(blk.data(), G, c->page);
        d2[i] = x.d; e2[i] = x.e;
      }
      bool found = false;
      for (u32 i = 0; i < cl.nb && !found; ++i) if (d2[i] != cl.d[i] || e2[i] != cl.e[i]) { bad = i; found = true; }
      ok = !found && chain_of(id, d2.data(), cl.nb) == cl.chain;
    }
    v[k].flags = V_SERVED | (ok ? V_OK : 0);
    v[k].bad = bad;
  }
}

// phase 2: per served claim, batch order: RESTORE_REQUIRED, then the outcome of the (merged) verdict; blocks of failed
// claims are freed.  request_id == 0: every claim is its own reuse request (blocking_claim_ids=[C]).  request_id
// != 0 (NEXT-3): the batch is ONE reuse request naming several claims; its refusal is emitted once, after the per-claim
// records, as one REFUSED record per failed claim (claim_id = the blocking claim, aux = REQ_FLAG | size of the failed
// subset, arg = request id) -- blocking_claim_ids is exactly the failed subset ("smeared" ids fail closed,
// P:L384).
static void restore_commit(Ctx* c, u32 n, const u64* ids, int32_t* st, const std::vector<Claim*>& served,
                           const std::vector<Verdict>& v, u64 request_id) {
  bool any_served = false;
  std::vector<u64> blocking;
  for (u32 k = 0; k < n; ++k) {
    if (!served[k]) continue;
    any_served = true;
    Claim& cl = *served[k]; u64 id = ids[k];
    c->emit(id, EV_RESTORE_REQUIRED, cl.M, 0);          // lookup "hit"
    drop_host(c, cl);
    if (v[k].flags & V_OK) {
      cl.state = CS_RESIDENT_AGAIN;
      c->emit(id, EV_RESTORED, cl.nb, c->tp_ranks > 1 ? 0 : cl.chain);
      st[k] = ST_OK;
    } else {
      c->emit(id, EV_LOAD_FAILED, v[k].bad, 0);
      c->emit(id, EV_RESTORATION_FAILED, 0, 0);
      if (cl.policy == POL_DEMOTE) c->emit(id, EV_DEMOTED, 0, 0);        // ordered responsibility boundary
      else if (cl.policy == POL_EXPIRE) c->emit(id, EV_EXPIRED, 0, 0);
      else if (request_id == 0) c->emit(id, EV_ACTIVE_REQUEST_REFUSED, 1, id);    // blocking_claim_ids=[C]: aux = count, arg = C
      else blocking.push_back(id);
      for (u32 b : cl.bt) { c->used[b] = 0; c->ref[b] = 0; c->fill[b] = 0; }
      cl.bt.clear(); cl.d.clear(); cl.e.clear();
      cl.state = cl.policy == POL_DEMOTE ? CS_DEMOTED : (cl.policy == POL_EXPIRE ? CS_EXPIRED : CS_REFUSED);   // terminal
      st[k] = ST_RESTORE_FAILED;
    }
  }
  for (u64 b : blocking) c->emit(b, EV_ACTIVE_REQUEST_REFUSED, REQ_FLAG | (u32)blocking.size(), request_id);
  if (any_served && (c->fault_flags & FF_ALLOW_UNCLAIMED)) {   // P:L337; generic counter only
    for (size_t f = 0; f < c->faults.size();)
      if (c->faults[f].claim_id == 0) { c->generic_failures++; c->faults.erase(c->faults.begin() + f); }
      else ++f;
  }
}

static void do_restore(Ctx* c, u32 n, const u64* ids, int32_t* st, u64 request_id = 0) {
  std::vector<Claim*> served;
  std::vector<Verdict> v;
  restore_verify(c, n, ids, st, served, v);
  restore_commit(c, n, ids, st, served, v, request_id);
}

// ---- NEXT-4: TP-sharded KV, one common verdict (DESIGN.md 8 / R24) ----------------------------------
// The pool is split by kv_head over G ranks; every rank makes the same calls on its own shard, with its own digests and
// chain.  The verdict must be common (attribution must survive; it must not smear): between phase 1 and
// phase 2 the ranks exchange their local verdicts, and every rank applies the SAME merged verdict per claim:
//   served  -- must agree on every rank (same calls, same allocator state); a disagreement is a call-level error;
//   ok      = AND over ranks;      bad = min over the ranks that failed (a transfer error, 0xFFFFFFFF, loses to a block index).
// In TP mode OFFLOADED / RESTORED carry arg = 0 (chains are rank-local facts; rco_claim_info still returns them), so the
// emitted streams are byte-identical on every rank.
static int tp_merge(u32 n, u32 G, const Verdict* gathered /*[G][n]*/, std::vector<Verdict>& out) {
  out.assign(n, Verdict{0, 0xFFFFFFFFu});
  for (u32 k = 0; k < n; ++k) {
    u32 served = gathered[k].flags & V_SERVED, ok = V_OK, bad = 0xFFFFFFFFu;
    for (u32 r = 0; r < G; ++r) {
      const Verdict& x = gathered[(u64)r * n + k];
      if ((x.flags & V_SERVED) != served) return E_INVALID;     // the ranks did not make the same call
      if (!(x.flags & V_OK)) { ok = 0; if (x.bad < bad) bad = x.bad; }
    }
    out[k].flags = served | (served ? ok : 0);
    out[k].bad = ok ? 0xFFFFFFFFu : bad;
  }
  return E_OK;
}

// ---- NEXT-3: allocator-side protection (reading R23) ------------------------------------------------
// P:L85 victim_exclusion_before_violation ("without victim exclusion, hard protection collapses to soft priority
// under pressure unless another explicit contract transition occurs first"), explicit_conflict_action,
// blocking_claim_ids, claim_demoted_before_loss; P:L103 hard_protected bundle; P:L270 allocator_hook ("exposes the
// victim candidate set, protected resident footprint, and ordered exclusion or release before predicate-breaking
// loss").  make_room(R, need): an active request R needs `need` free blocks.
//   1. F = free blocks.  F >= need: OK, nothing happens.
//   2. Victim candidates = live claims that hold a table (ACCEPTED, MATERIALIZED, RESIDENT_AGAIN): the unprotected
//      ones first, then the protected ones, each group in acceptance order.  Evicting a claim frees the blocks whose
//      last reference it holds.  m = the shortest prefix of the list whose eviction brings the free count to `need`.
//   3. m exists and lies inside the unprotected group: those m claims are demoted, in list order -- DEMOTED(C,
//      aux = table blocks released, arg = R) is emitted BEFORE the claim's references are dropped (ordered release
//      before loss); state DEMOTED (terminal).  Status OK; ids = the demoted claims.
//   4. otherwise the need could only be met from a protected footprint: NOTHING is evicted, no block changes hands.
//      If protected candidates exist, the request is refused: one CONFLICT_REFUSED record per blocking claim, in list
//      order, claim_id = the blocking claim, aux = REQ_FLAG | k, arg = R; blocking_claim_ids = the k protected claims
//      the walk had to enter (all of them if even that is not enough).  Status PROTECTED_CONFLICT; ids = those claims.
//      With no protected candidate: NO_FREE_BLOCKS, no event.
static int do_make_room(Ctx* c, u64 request_id, u32 need, u64* ids_out, u32 cap, u32* n_out) {
  *n_out = 0;
  u64 nfree = 0;
  for (u32 b = 0; b < c->NB; ++b) nfree += !c->used[b];
  if (nfree >= need) return ST_OK;
  std::vector<std::pair<u64, u64>> cand[2];             // (acceptance order, id); [0] unprotected, [1] protected
  for (auto& kv : c->claims) {
    const Claim& cl = kv.second;
    if (cl.state == CS_ACCEPTED || cl.state == CS_MATERIALIZED || cl.state == CS_RESIDENT_AGAIN)
      cand[cl.protect ? 1 : 0].push_back({cl.order, kv.first});
  }
  std::sort(cand[0].begin(), cand[0].end()); std::sort(cand[1].begin(), cand[1].end());
  std::vector<u64> list;
  for (auto& x : cand[0]) list.push_back(x.second);
  const size_t U = list.size();
  for (auto& x : cand[1]) list.push_back(x.second);
  std::vector<u32> ref = c->ref;                         // trial walk on a copy: nothing is evicted yet
  size_t m = 0; bool met = false;
  u64 f = nfree;
  while (m < list.size()) {
    for (u32 b : c->claims[list[m]].bt) if (--ref[b] == 0) ++f;
    ++m;
    if (f >= need) { met = true; break; }
  }
  if (met && m <= U) {
    for (size_t k = 0; k < m; ++k) {
      Claim& cl = c->claims[list[k]];
      c->emit(list[k], EV_DEMOTED, (u32)cl.bt.size(), request_id);   // the boundary precedes the loss
      drop_refs(c, cl);
      cl.state = CS_DEMOTED;
      if (*n_out < cap) ids_out[*n_out] = list[k];
      ++*n_out;
    }
    return ST_OK;
  }
  if (list.size() == U) return ST_NO_FREE_BLOCKS;       // no protected footprint is in the way: plain exhaustion
  const size_t hi = met ? m : list.size();
  const u32 k = (u32)(hi - U);
  for (size_t i = U; i < hi; ++i) {
    c->emit(list[i], EV_CONFLICT_REFUSED, REQ_FLAG | k, request_id);
    if (*n_out < cap) ids_out[*n_out] = list[i];
    ++*n_out;
  }
  return ST_PROTECTED_CONFLICT;
}

// ---- C ABI (host pointers everywhere) ---------------------------------------
struct rco_config { u32 layers, kv_heads, head_dim, elem_bytes, block_size, pool_blocks;
                    u64 host_store_bytes; void* pool; u8* fill; };

extern "C" {

int rco_create(const rco_config* cfg, void** out) {
  if (!cfg || !out || !cfg->pool || !cfg->fill) return E_INVALID;
  u64 page = (u64)cfg->block_size * cfg->kv_heads * cfg->head_dim * cfg->elem_bytes;
  if (page == 0 || page % 4096 != 0 || cfg->layers == 0 || cfg->pool_blocks == 0) return E_INVALID;
  Ctx* c = new Ctx();
  c->L = cfg->layers; c->H = cfg->kv_heads; c->D = cfg->head_dim; c->e = cfg->elem_bytes;
  c->BS = cfg->block_size; c->NB = cfg->pool_blocks; c->page = page; c->blk = 2ull * c->L * page;
  c->host_cap = cfg->host_store_bytes; c->pool = (u8*)cfg->pool; c->fill = cfg->fill;
  c->used.assign(c->NB, 0); c->ref.assign(c->NB, 0);
  *out = c; return E_OK;
}
int rco_destroy(void* h) { delete (Ctx*)h; return E_OK; }

int rco_mark_used(void* h, u32 n, const u32* ids) {
  Ctx* c = (Ctx*)h;
  for (u32 i = 0; i < n; ++i) if (ids[i] >= c->NB) return E_INVALID;
  for (u32 i = 0; i < n; ++i) c->used[ids[i]] = 1;
  return E_OK;
}
int rco_mark_free(void* h, u32 n, const u32* ids) {      // claimed blocks (ref>0) are left alone
  Ctx* c = (Ctx*)h;
  for (u32 i = 0; i < n; ++i) if (ids[i] >= c->NB) return E_INVALID;
  for (u32 i = 0; i < n; ++i) if (c->ref[ids[i]] == 0) c->used[ids[i]] = 0;
  return E_OK;
}
int rco_accept(void* h, u32 n, const u64* id, const u32* P, const u32* N, const u32* bt_off,
               const u32* bt_ids, int32_t* st) {
  Ctx* c = (Ctx*)h;
  for (u32 k = 0; k < n; ++k) {
    if (bt_off[k + 1] < bt_off[k]) { st[k] = ST_BAD_TABLE; continue; }
    st[k] = do_accept(c, id[k], P[k], N[k], bt_ids + bt_off[k], bt_off[k + 1] - bt_off[k]);
  }
  return E_OK;
}
int rco_materialize(void* h, u32 n, const u64* id, int32_t* st) {
  for (u32 k = 0; k < n; ++k) st[k] = do_materialize((Ctx*)h, id[k]);
  return E_OK;
}
int rco_offload(void* h, u32 n, const u64* id, int32_t* st) { do_offload((Ctx*)h, n, id, st); return E_OK; }
int rco_restore(void* h, u32 n, const u64* id, int32_t* st) { do_restore((Ctx*)h, n, id, st); return E_OK; }
int rco_restore_request(void* h, u64 request_id, u32 n, const u64* id, int32_t* st) {
  if (request_id == 0) return E_INVALID;
  do_restore((Ctx*)h, n, id, st, request_id); return E_OK;
}
int rco_set_policy(void* h, u32 n, const u64* id, const u32* policy) {   // what a failed restoration means for the claim
  Ctx* c = (Ctx*)h;
  for (u32 k = 0; k < n; ++k) if (!c->claims.count(id[k]) || policy[k] > POL_EXPIRE) return E_INVALID;
  for (u32 k = 0; k < n; ++k) c->claims[id[k]].policy = policy[k];
  return E_OK;
}
int rco_set_tp(void* h, u32 ranks) { ((Ctx*)h)->tp_ranks = ranks; return E_OK; }
int rco_tp_restore_verify(void* h, u32 n, const u64* id, int32_t* st, Verdict* local) {
  Ctx* c = (Ctx*)h;
  if (c->tp_pending || c->dedup) return E_INVALID;
  std::vector<Claim*> served; std::vector<Verdict> v;
  restore_verify(c, n, id, st, served, v);
  for (u32 k = 0; k < n; ++k) { local[k] = v[k]; if (served[k]) st[k] = -1; }   // pending: decided by the commit
  c->tp_ids.assign(id, id + n);
  c->tp_served.assign(served.begin(), served.end());
  c->tp_pending = true;
  return E_OK;
}
int rco_tp_restore_commit(void* h, u32 n, u32 G, const Verdict* gathered, int32_t* st) {
  Ctx* c = (Ctx*)h;
  if (!c->tp_pending || n != c->tp_ids.size() || G == 0) return E_INVALID;
  std::vector<Verdict> merged;
  if (tp_merge(n, G, gathered, merged) != E_OK) return E_INVALID;
  std::vector<Claim*> served(n);
  for (u32 k = 0; k < n; ++k) {
    served[k] = (Claim*)c->tp_served[k];
    if (((merged[k].flags & V_SERVED) != 0) != (served[k] != nullptr)) return E_INVALID;
  }
  restore_commit(c, n, c->tp_ids.data(), st, served, merged, 0);
  c->tp_pending = false;
  return E_OK;
}
// Split form of restore (rc.h rc_restore_begin / rc_wait(1); reading R25): the same two phases that
// rco_restore runs back to back, with other calls allowed in between -- phase 1 (eligibility, grant, allocation, fault
// decision, write, re-digest, verdict) at _begin, phase 2 (RESTORE_REQUIRED and the outcome records, release of the host
// copy, release of the blocks of failed claims) at _end.  No arithmetic of its own.
int rco_restore_begin(void* h, u64 request_id, u32 n, const u64* id, int32_t* st) {
  Ctx* c = (Ctx*)h;
  if (c->tp_pending) return E_INVALID;
  std::vector<Claim*> served;
  restore_verify(c, n, id, st, served, c->split_v);
  for (u32 k = 0; k < n; ++k) if (served[k]) { st[k] = -1; served[k]->in_flight = true; }   // pending: decided by _end
  c->tp_ids.assign(id, id + n);
  c->tp_served.assign(served.begin(), served.end());
  c->split_request = request_id;
  c->tp_pending = true;
  return E_OK;
}
int rco_restore_end(void* h, int32_t* st) {
  Ctx* c = (Ctx*)h;
  if (!c->tp_pending) return E_INVALID;
  const u32 n = (u32)c->tp_ids.size();
  std::vector<Claim*> served(n);
  for (u32 k = 0; k < n; ++k) { served[k] = (Claim*)c->tp_served[k]; if (served[k]) served[k]->in_flight = false; }
  restore_commit(c, n, c->tp_ids.data(), st, served, c->split_v, c->split_request);
  c->tp_pending = false;
  return E_OK;
}
int rco_protect(void* h, u32 n, const u64* id, const u32* on) {          // hard_protected on / off; any live claim
  Ctx* c = (Ctx*)h;
  for (u32 k = 0; k < n; ++k) {
    auto it = c->claims.find(id[k]);
    if (it == c->claims.end() || on[k] > 1 || it->second.state >= CS_REFUSED) return E_INVALID;
  }
  for (u32 k = 0; k < n; ++k) c->claims[id[k]].protect = on[k];
  return E_OK;
}
int rco_make_room(void* h, u64 request_id, u32 need, int32_t* status, u64* ids, u32 cap, u32* n_ids) {
  if (request_id == 0 || !status || !n_ids) return E_INVALID;
  *status = do_make_room((Ctx*)h, request_id, need, ids, cap, n_ids);
  return E_OK;
}
int rco_protected_map(void* h, u8* prot) {               // prot[NB]: 1 = block lies in a protected footprint
  Ctx* c = (Ctx*)h;
  memset(prot, 0, c->NB);
  for (auto& kv : c->claims) if (kv.second.protect) for (u32 b : kv.second.bt) prot[b] = 1;
  return E_OK;
}
int rco_release(void* h, u32 n, const u64* id, int32_t* st) {
  Ctx* c = (Ctx*)h;
  for (u32 k = 0; k < n; ++k) {
    auto it = c->claims.find(id[k]);
    if (it == c->claims.end()) { st[k] = ST_UNKNOWN_CLAIM; continue; }
    if (it->second.in_flight) { st[k] = ST_BAD_STATE; continue; }   // a claim of a restore in flight (rc.h)
    drop_refs(c, it->second);
    drop_host(c, it->second);
    c->claims.erase(it); st[k] = ST_OK;
  }
  return E_OK;
}
int rco_outcomes(void* h, Event* buf, u64 cap, u64* n_out) {
  Ctx* c = (Ctx*)h; u64 k = 0;
  while (k < cap && c->drained < c->events.size()) buf[k++] = c->events[c->drained++];
  *n_out = k; return E_OK;
}
int rco_set_faults(void* h, u32 n, const Fault* f, u32 flags) {
  Ctx* c = (Ctx*)h;
  for (u32 i = 0; i < n; ++i) {
    if (f[i].kind != FK_XFER_ERROR && f[i].kind != FK_BITFLIP) return E_INVALID;
    if (f[i].claim_id == 0 && !(flags & FF_ALLOW_UNCLAIMED)) return E_INVALID;  // P:L337 separate flag
  }
  c->faults.assign(f, f + n); c->fault_flags = flags;
  return E_OK;
}
int rco_claim_info(void* h, u64 id, ClaimInfo* o) {
  Ctx* c = (Ctx*)h; auto it = c->claims.find(id);
  if (it == c->claims.end()) return E_INVALID;
  const Claim& cl = it->second;
  o->claim_id = id; o->chain = cl.chain; o->host_bytes = host_size_of(c, cl); o->state = cl.state;
  o->P = cl.P; o->N = cl.N; o->M = cl.M; o->nb = cl.nb; o->n_table = (u32)cl.bt.size();
  return E_OK;
}
int rco_claim_blocks(void* h, u64 id, u32* ids, u32 cap, u32* n) {
  Ctx* c = (Ctx*)h; auto it = c->claims.find(id);
  if (it == c->claims.end()) return E_INVALID;
  *n = (u32)it->second.bt.size();
  for (u32 i = 0; i < *n && i < cap; ++i) ids[i] = it->second.bt[i];
  return E_OK;
}
int rco_claim_digests(void* h, u64 id, u64* d, u64* e, u32 cap, u32* n) {   // e may be NULL
  Ctx* c = (Ctx*)h; auto it = c->claims.find(id);
  if (it == c->claims.end()) return E_INVALID;
  *n = (u32)it->second.d.size();
  for (u32 i = 0; i < *n && i < cap; ++i) { d[i] = it->second.d[i]; if (e) e[i] = it->second.e[i]; }
  return E_OK;
}
int rco_host_read(void* h, u64 id, void* dst, u64 cap, u64* bytes) {
  Ctx* c = (Ctx*)h; auto it = c->claims.find(id);
  if (it == c->claims.end()) return E_INVALID;
  const std::vector<u8> hb = host_bytes_of(c, it->second);
  *bytes = hb.size();
  if (dst && cap >= *bytes && *bytes) memcpy(dst, hb.data(), *bytes);
  return E_OK;
}
int rco_pool_state(void* h, u8* used, u32* ref) {       // copies used[NB], ref[NB]
  Ctx* c = (Ctx*)h;
  if (used) memcpy(used, c->used.data(), c->NB);
  if (ref) memcpy(ref, c->ref.data(), 4ull * c->NB);
  return E_OK;
}
int rco_stats(void* h, u64* out4) {                     // host_used, n_claims, n_events, generic_failures
  Ctx* c = (Ctx*)h;
  out4[0] = c->host_used; out4[1] = c->claims.size(); out4[2] = c->events.size(); out4[3] = c->generic_failures;
  return E_OK;
}
int rco_set_dedup(void* h, int on) {                    // only while no claim holds host bytes
  Ctx* c = (Ctx*)h;
  if (c->host_used != 0 || (on && c->layer_major)) return E_INVALID;
  c->dedup = on != 0; return E_OK;
}
int rco_set_layer_major(void* h, int on) {              // only while no claim holds host bytes; not with dedup
  Ctx* c = (Ctx*)h;
  if (c->host_used != 0 || c->dedup) return E_INVALID;
  c->layer_major = on != 0; return E_OK;
}
int rco_link_bytes(void* h, u64* out2) { Ctx* c = (Ctx*)h; out2[0] = c->link_d2h; out2[1] = c->link_h2d; return E_OK; }
// checksum primitives, exported so the pins can reach each one directly
u64 rco_mixL(u64 x) { return mixL(x); }
u64 rco_mixF(u64 x) { return mixF(x); }
u64 rco_mum(u64 x, u64 y) { return mum(x, y); }
// which: 0 = the checksum family (d), 1 = the key-extension family (e)
u64 rco_page_digest(const void* p, u64 page_bytes, int which) { Dig2 x = page_digest2((const u8*)p, page_bytes); return which ? x.e : x.d; }
u64 rco_block_digest(const void* p, u32 n_pages, u64 page_bytes, int which) {
  Dig2 x = block_digest2((const u8*)p, n_pages, page_bytes); return which ? x.e : x.d;
}
u64 rco_chain_of(u64 id, const u64* d, u32 nb) { return chain_of(id, d, nb); }

}  // extern "C"
