// rc_trace.cuh -- NEXT-1: the paper's artifact analyzer ("supplies no runtime
// behavior; it only checks order, claim match, and controls after the run") as a data-parallel pass over
// an event array.  Events are grouped by claim with a device hash table (no global sort), every claim's
// subsequence is replayed through the per-claim automaton of DESIGN.md "Validator" by one thread, and the
// first violating stream position is a min-reduction.  Rules and passages:
//   seq strictly increasing; an event naming no claim (id 0) is invalid;
//   nothing names a claim before its ACCEPTED;
//   USE(C) while C is offloaded / restore-required is invalid: restore-after-use;
//   REQUEST_FINISHED(C) between LOAD_FAILED and REFUSED is invalid: outcome precedes terminal handling;
//   LOAD_FAILED / RESTORATION_FAILED / REFUSED without RESTORE_REQUIRED(C) in the same cycle is invalid;
//   REFUSED must carry blocking_claim_ids = [C] (aux 1, arg C).
// Allocator-side protection (NEXT-3): DEMOTED(C, arg = request id != 0) while C is resident is
// the ordered demotion of a victim before its blocks are lost (after RESTORATION_FAILED, DEMOTED keeps arg = 0);
// CONFLICT_REFUSED(C, aux = REQ_FLAG | k, arg = request id != 0) names a resident claim that blocks an active request;
// the k records of one refusal are consecutive and name k different claims.
#pragma once
#include "rc_kernels.cuh"

namespace rct {
using namespace rck;

enum { S0 = 0, ACC, MAT, OFF, RREQ, LF, RF, REF, RES, FIN, DEM, EXP, BAD, NSTATE };
enum { EV_USE = 100, EV_FIN = 101 };
enum { G_FAILURE = 1, G_OBSERVATION = 2 };
constexpr u64 NO_BAD = ~0ull;

struct ClaimOut { u64 claim_id; u64 first_bad; u32 state; u32 gates; u32 n_events; u32 pad; };

__device__ __forceinline__ int col_of(u32 code) {
  return code >= 1 && code <= 8 ? (int)code - 1 : (code == EV_USE ? 8 : (code == EV_FIN ? 9 : (code == EV_DEMOTED ? 10 : (code == EV_EXPIRED ? 11 : (code == EV_CONFLICT_REFUSED ? 12 : -1)))));
}

// next-state table [state][column]; BAD = not in the accepted language
__device__ __forceinline__ u32 next_state(u32 s, int col) {
  // columns: 0 ACCEPTED 1 MATERIALIZED 2 OFFLOADED 3 RESTORE_REQUIRED 4 LOAD_FAILED 5 RESTORED 6 RESTORATION_FAILED 7 REFUSED 8 USE 9 FIN
  //          10 DEMOTED 11 EXPIRED 12 CONFLICT_REFUSED (NEXT-3)
  switch (s) {
    case S0:   return col == 0 ? ACC : BAD;
    case ACC:  return col == 1 ? MAT : (col == 9 ? FIN : (col == 10 ? DEM : (col == 12 ? ACC : BAD)));
    case MAT:  return col == 2 ? OFF : (col == 8 ? MAT : (col == 9 ? FIN : (col == 10 ? DEM : (col == 12 ? MAT : BAD))));
    case OFF:  return col == 3 ? RREQ : BAD;
    case RREQ: return col == 5 ? RES : (col == 4 ? LF : BAD);
    case LF:   return col == 6 ? RF : BAD;
    case RF:   return col == 7 ? REF : (col == 10 ? DEM : (col == 11 ? EXP : BAD));
    case REF:  return col == 9 ? FIN : BAD;
    case DEM:  return col == 9 ? FIN : BAD;
    case EXP:  return col == 9 ? FIN : BAD;
    case RES:  return col == 2 ? OFF : (col == 8 ? RES : (col == 9 ? FIN : (col == 10 ? DEM : (col == 12 ? RES : BAD))));
    default:   return BAD;
  }
}

__device__ __forceinline__ u64 hash64(u64 x) { return mixF(x); }

// pass 1: stream-level checks, hash insert, per-slot event count
__global__ void tv_insert(const Event* __restrict__ ev, u64 n, u64* __restrict__ keys, u32* __restrict__ count, u32 mask,
                          u32* __restrict__ slot_of, unsigned long long* __restrict__ first_bad) {
  const u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const Event e = ev[i];
  if (i > 0 && e.seq <= ev[i - 1].seq) atomicMin(first_bad, (unsigned long long)i);
  if (e.claim_id == 0) { atomicMin(first_bad, (unsigned long long)i); slot_of[i] = 0xFFFFFFFFu; return; }
  u32 h = (u32)hash64(e.claim_id) & mask;
  for (;;) {
    const u64 k = keys[h];
    if (k == e.claim_id) break;
    if (k == 0) {
      const u64 old = atomicCAS((unsigned long long*)&keys[h], 0ull, (unsigned long long)e.claim_id);
      if (old == 0 || old == e.claim_id) break;
    }
    h = (h + 1) & mask;
  }
  slot_of[i] = h;
  atomicAdd(&count[h], 1u);
}

// pass 2: bucket space and a dense claim index per occupied slot
__global__ void tv_alloc(const u32* __restrict__ count, u32 slots, u32* __restrict__ base, u32* __restrict__ dense,
                         u32* __restrict__ cursors /*[0] events, [1] claims*/) {
  const u32 s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= slots || count[s] == 0) return;
  base[s] = atomicAdd(&cursors[0], count[s]);
  dense[s] = atomicAdd(&cursors[1], 1u);
}

// pass 3: event indices into their claim's bucket (arrival order is arbitrary; pass 4 orders them)
__global__ void tv_scatter(u64 n, const u32* __restrict__ slot_of, const u32* __restrict__ base, u32* __restrict__ fill,
                           u32* __restrict__ bucket) {
  const u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const u32 s = slot_of[i];
  if (s == 0xFFFFFFFFu) return;
  bucket[base[s] + atomicAdd(&fill[s], 1u)] = (u32)i;
}

// pass 4: one thread per claim: order its events by stream position, replay the automaton, derive the gates
__global__ void tv_walk(const Event* __restrict__ ev, const u64* __restrict__ keys, const u32* __restrict__ count, u32 slots,
                        const u32* __restrict__ base, const u32* __restrict__ dense, u32* __restrict__ bucket,
                        ClaimOut* __restrict__ out, unsigned long long* __restrict__ first_bad) {
  const u32 s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= slots) return;
  const u32 c = count[s];
  if (c == 0) return;
  u32* b = bucket + base[s];
  if (c <= 16) {                                // a claim has a handful of events: insertion sort
    for (u32 i = 1; i < c; ++i) {
      const u32 x = b[i];
      u32 j = i;
      while (j > 0 && b[j - 1] > x) { b[j] = b[j - 1]; --j; }
      b[j] = x;
    }
  } else {                                      // a claim with many events (long USE runs, many cycles): heap sort, O(c log c)
    auto sift = [&](u32 root, u32 end) {
      for (;;) {
        u32 ch = 2 * root + 1;
        if (ch >= end) break;
        if (ch + 1 < end && b[ch + 1] > b[ch]) ++ch;
        if (b[root] >= b[ch]) break;
        const u32 t = b[root]; b[root] = b[ch]; b[ch] = t;
        root = ch;
      }
    };
    for (u32 i = c / 2; i-- > 0;) sift(i, c);
    for (u32 end = c - 1; end > 0; --end) { const u32 t = b[0]; b[0] = b[end]; b[end] = t; sift(0, end); }
  }
  const u64 cid = keys[s];
  u32 st = S0, n_codes = 0, c0 = 0, c1 = 0, tail = 0;   // tail: last five lifecycle codes, 4 bits each
  bool saw_fail = false;
  u64 bad = NO_BAD;
  u64 cr_arg = 0; u32 cr_aux = 0, cr_pos = 0; bool cr_any = false;   // the claim's last CONFLICT_REFUSED record
  for (u32 i = 0; i < c; ++i) {
    const Event e = ev[b[i]];
    const int col = col_of(e.code);
    u32 nx = col < 0 ? (u32)BAD : next_state(st, col);
    // DEMOTED: arg = 0 after a failed restoration, = the request id for a victim of rc_make_room
    if (nx != BAD && col == 10 && ((e.arg == 0) != (st == RF))) nx = BAD;
    if (nx != BAD && col == 12) {
      const u32 k = e.aux & ~REQ_FLAG;
      if (!(e.aux & REQ_FLAG) || k == 0 || e.arg == 0) nx = BAD;
      else if (cr_any && cr_arg == e.arg && cr_aux == e.aux && b[i] - cr_pos < k) nx = BAD;   // named twice in one run
      cr_any = true; cr_arg = e.arg; cr_aux = e.aux; cr_pos = b[i];
    }
    // per-claim refusal carries [C] itself; the request form (REQ_FLAG) is checked across claims by tv_groups
    if (nx != BAD && e.code == EV_ACTIVE_REQUEST_REFUSED && !(e.aux & REQ_FLAG) && (e.arg != cid || e.aux != 1)) nx = BAD;
    if (nx == BAD) { bad = b[i]; st = BAD; break; }
    st = nx;
    if (col < 8 || col == 10 || col == 11) {
      if (n_codes == 0) c0 = e.code; else if (n_codes == 1) c1 = e.code;
      tail = ((tail << 4) | e.code) & 0xFFFFFu;
      ++n_codes;
      saw_fail |= (e.code == EV_LOAD_FAILED || e.code == EV_ACTIVE_REQUEST_REFUSED);
    }
  }
  u32 gates = 0;
  if (bad == NO_BAD && c0 == EV_ACCEPTED && c1 == EV_MATERIALIZED) {
    // failure gate: subsequence ends OFFLOADED RESTORE_REQUIRED LOAD_FAILED RESTORATION_FAILED REFUSED
    if (n_codes >= 7 && tail == 0x34578u) gates |= G_FAILURE;
    // observation gate: ends OFFLOADED RESTORE_REQUIRED RESTORED, no failure record names C
    if (n_codes >= 5 && (tail & 0xFFFu) == 0x346u && !saw_fail) gates |= G_OBSERVATION;
  }
  if (bad != NO_BAD) atomicMin(first_bad, (unsigned long long)bad);
  out[dense[s]] = ClaimOut{cid, bad, st, gates, c, 0};
}

// ---- request-level refusal runs (NEXT-3) -----------------------------------------------------
// pending(i) = claims whose restoration failed and is unanswered before stream position i
//            = #RESTORATION_FAILED - #(REFUSED | DEMOTED | EXPIRED) among events [0, i)   (valid up to the first violation).
__device__ __forceinline__ u32 pend_delta(const Event& e) {
  return e.code == EV_RESTORATION_FAILED ? 1u
       : ((e.code == EV_ACTIVE_REQUEST_REFUSED || (e.code == EV_DEMOTED && e.arg == 0) || e.code == EV_EXPIRED) ? 0xFFFFFFFFu : 0u);
}
__global__ void tv_delta_sum(const Event* __restrict__ ev, u64 n, u32* __restrict__ bsum) {
  __shared__ u32 wt[32];
  const u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x;
  u32 tot;
  block_scan_incl(i < n ? pend_delta(ev[i]) : 0u, wt, tot);
  if (threadIdx.x == 0) bsum[blockIdx.x] = tot;
}
__global__ void tv_scan_bsum(u32* __restrict__ bsum, u32 nb) {          // exclusive scan in place, one CTA
  __shared__ u32 wt[32];
  u32 carry = 0;
  for (u32 base = 0; base < nb; base += blockDim.x) {
    const u32 k = base + threadIdx.x;
    const u32 v = k < nb ? bsum[k] : 0u;
    u32 tot;
    const u32 inc = block_scan_incl(v, wt, tot);
    if (k < nb) bsum[k] = carry + inc - v;
    carry += tot;
    __syncthreads();
  }
}
__device__ __forceinline__ bool same_run(const Event& a, u32 code, u64 arg, u32 aux) {
  return a.code == code && a.arg == arg && a.aux == aux;
}
// A run of REFUSED records with the same (arg = request id, aux = REQ_FLAG | k) starts where the previous record does
// not match.  The start checks: k >= 1 and k == pending (the run names exactly the failed, unanswered claims: neither
// fewer nor -- via the per-claim automaton -- others); records 1..k-1 continue the run; a matching record at k would
// open a second run with nothing pending.
__global__ void tv_groups(const Event* __restrict__ ev, u64 n, const u32* __restrict__ boff, unsigned long long* __restrict__ first_bad) {
  __shared__ u32 wt[32];
  const u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x;
  Event e; e.code = 0; e.aux = 0; e.arg = 0;
  if (i < n) e = ev[i];
  const u32 d = i < n ? pend_delta(e) : 0u;
  u32 tot;
  const u32 pending = boff[blockIdx.x] + block_scan_incl(d, wt, tot) - d;
  const bool conflict = e.code == EV_CONFLICT_REFUSED;                   // same run shape, no pending rule
  if (i >= n || !(e.code == EV_ACTIVE_REQUEST_REFUSED || conflict) || !(e.aux & REQ_FLAG)) return;
  if (i > 0 && same_run(ev[i - 1], e.code, e.arg, e.aux)) return;        // not a run start
  const u32 k = e.aux & ~REQ_FLAG;
  if (k == 0 || (!conflict && k != pending)) { atomicMin(first_bad, (unsigned long long)i); return; }
  for (u32 j = 1; j < k && i + j < n; ++j)
    if (!same_run(ev[i + j], e.code, e.arg, e.aux)) { atomicMin(first_bad, (unsigned long long)(i + j)); return; }
  if (i + k < n && same_run(ev[i + k], e.code, e.arg, e.aux)) atomicMin(first_bad, (unsigned long long)(i + k));
}

}  // namespace rct
