// rc_kernels.cuh -- device code of librc (sm_100a only).
//
// Kernels of the claim-scoped KV offload / restore path:
//   k_pred          K1  leading-prefix-at-least-N from fill[] (warp ballot + ffs)
//   k_offsets       K1  exclusive scan of per-claim block counts (block scan)
//   k_worklist      K1  compacted physical-block list (warp per claim)
//   k_move_hash     K2/K4 page gather / scatter with the lane-fold checksum fused in   BJ (b),(c),(d)
//   k_move_hash_tma K2/K4 same, staged through cp.async.bulk (TMA) + mbarrier ring
//   k_block_digest  K2/K4 tail: page terms -> per-block digest
//   k_chain         K3  per-claim affine warp scan of block digests                     BJ (d)
//   k_restore_plan  K5  free count, prefix grant, lowest-free-id allocation             DESIGN R6/R7
//   k_verify        K4/K3 digest compare, chain compare, verdict, fill / free
//   k_unref         K5  reference drop at offload
//   k_accept        a0  table validation + reference take
//   k_emit          K6  ordered claim-scoped event records (scan-assigned offsets)
// The checksum constants are restated here from DESIGN.md "Checksum"; nothing is
// shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

typedef uint64_t u64;
typedef uint32_t u32;
typedef uint8_t u8;

namespace rck {

constexpr u64 C1 = 0x9E3779B97F4A7C15ull;
constexpr u64 C2 = 0x6A09E667F3BCC909ull;
constexpr u64 CA = 0xBB67AE8584CAA73Bull;
constexpr u64 C3 = 0x3C6EF372FE94F82Bull;
constexpr u64 C4 = 0xA54FF53A5F1D36F1ull;
constexpr u64 C5 = 0x510E527FADE682D1ull;
constexpr u32 SKIP = 0xFFFFFFFFu;       // work item whose transfer was suppressed (XFER_ERROR)
constexpr int LANES = 256;              // checksum lanes per page == threads per CTA of k_move_hash
constexpr int WPC = LANES / 32;         // warps per CTA

// batch descriptor, one per claim of a call (host fills, device reads)
struct Desc {
  u64 id, chain;
  u32 P, N, M, nb;
  u32 bt_off, bt_len;     // table extent in the arena (bt_len entries)
  u32 dg_off;             // digest extent in the digest arena (nb entries)
  u32 flags;              // D_* below
  u32 src_off;            // accept: offset of the candidate table in the upload buffer
  u32 pad;                // restore: the claim's failure policy (POL_*)
};
enum { D_ELIG = 1, D_XFER = 2, D_PROT = 4 };

// per-claim result of a call (device fills, host reads)
struct Res {
  u32 flag;               // R_* below
  u32 val;                // M (materialize) or first bad block (restore)
  u64 chain;
};
enum { R_OK = 1, R_SERVED = 2 };

struct Event { u64 seq, claim_id; u32 code, aux; u64 arg; };
enum { EV_ACCEPTED = 1, EV_MATERIALIZED = 2, EV_OFFLOADED = 3, EV_RESTORE_REQUIRED = 4, EV_LOAD_FAILED = 5,
       EV_RESTORED = 6, EV_RESTORATION_FAILED = 7, EV_ACTIVE_REQUEST_REFUSED = 8 };
enum { EM_ACCEPT = 0, EM_MATERIALIZE = 1, EM_OFFLOAD = 2, EM_RESTORE = 3, EM_DEMOTE = 4, EM_CONFLICT = 5 };
enum { EV_CONFLICT_REFUSED = 11 };                   // NEXT-3: active_request_refused(blocking_claim_ids) under hard protection
enum { VO_FITS = 0, VO_EVICT = 1, VO_CONFLICT = 2, VO_NOFREE = 3 };   // outcome of k_vic_decide
enum { EV_DEMOTED = 9, EV_EXPIRED = 10 };            // NEXT-3: other claim-scoped outcomes of a failed restoration
enum { POL_REFUSE = 0, POL_DEMOTE = 1, POL_EXPIRE = 2 };   // Desc.pad carries the claim's failure policy
constexpr u32 REQ_FLAG = 0x80000000u;                // REFUSED.aux of a request-level refusal: flag | subset size

__device__ __forceinline__ u64 mixL(u64 x) { u64 y = x ^ (x >> 32); y *= C2; return y ^ (y >> 29); }
__device__ __forceinline__ u64 mixF(u64 x) { u64 y = mixL(x); y *= C1; return y ^ (y >> 32); }

__device__ __forceinline__ u64 shfl_xor64(u64 v, int m) { return __shfl_xor_sync(0xFFFFFFFFu, v, m); }
__device__ __forceinline__ u64 shfl_up64(u64 v, int d) { return __shfl_up_sync(0xFFFFFFFFu, v, d); }
__device__ __forceinline__ u64 warp_sum64(u64 v) {
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) v += shfl_xor64(v, m);
  return v;
}
__device__ __forceinline__ u32 warp_sum32(u32 v) {
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, m);
  return v;
}

// streaming 16-byte accesses: the data is touched once, keep it out of L1 and first out of L2
__device__ __forceinline__ uint4 ld_stream(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_stream(uint4* p, const uint4& v) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};"
               :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
// DESIGN.md "Checksum" R22: one 16-byte vector (a, b) per step, two independent lane families.
//   h = mum(a ^ C2, b ^ h)   (the checksum d)        g = mum(b ^ C5, a ^ g)   (the key extension e)
// mum = 128-bit product folded low ^ high: mul.lo.u64 + mul.hi.u64 (4 IMAD.WIDE + carries each pair).
__device__ __forceinline__ u64 mum(u64 x, u64 y) { return (x * y) ^ __umul64hi(x, y); }
__device__ __forceinline__ void fold2(u64& h, u64& g, const uint4& v) {
  const u64 a = (u64)v.x | ((u64)v.y << 32), b = (u64)v.z | ((u64)v.w << 32);
  h = mum(a ^ C2, b ^ h);
  g = mum(b ^ C5, a ^ g);
}

// ---------------------------------------------------------------------------------------------
// K2 / K4: page mover with fused checksum.  One CTA (256 threads = the 256 checksum lanes) per
// page at a time, grid-stride over the n_items*G pages of a staging chunk.  Thread t moves
// vectors t, t+256, ... of the page (each warp access = 512 contiguous bytes) and folds them in
// that order; each warp writes the sums of its 32 lane terms (both families) to part[(page*8 + warp)*2 + {0,1}]
// -- no block barrier and no atomics in the streaming loop.  MODE 0 gather (pool -> staging), 1 scatter
// (staging -> pool), 2 digest only (read staging).  The staged position of page g of item w is w*sw + g*sg pages:
// (sw, sg) = (G, 1) is the block-major chunk [item][g][page]; (1, n_items) the layer-major chunk [g][item][page]
// (rc_config.layer_major, NEXT-4).  Partial sums are indexed by (item, g) either way, so the digests do not change.
// ---------------------------------------------------------------------------------------------
enum { MV_GATHER = 0, MV_SCATTER = 1, MV_DIGEST = 2 };

template <int MODE, int UNR>
__global__ void __launch_bounds__(LANES)
k_move_hash(uint4* __restrict__ pool, uint4* __restrict__ staging, const u32* __restrict__ phys,
            u64* __restrict__ part, u32 n_items, u32 G, u32 NB, u32 vpp,
            const u32* __restrict__ iw /*item -> work position (nullptr: identity)*/,
            const u32* __restrict__ ispos /*item -> staged block (nullptr: identity; NEXT-2 shared staging)*/,
            u32 sw, u32 sg /*staged page of (item w, page g) = w*sw + g*sg: (G, 1) block-major, (1, n_items) layer-major*/) {
  const u32 t = threadIdx.x;
  const u32 n_pages = n_items * G;
  const u32 vpt = vpp / LANES;
  for (u32 u = blockIdx.x; u < n_pages; u += gridDim.x) {
    const u32 w = u / G, g = u - w * G;
    u32 b = 0;
    if (MODE != MV_DIGEST) { b = __ldg(phys + (iw ? __ldg(iw + w) : w)); if (b == SKIP) continue; }
    uint4* pp = pool + ((u64)g * NB + b) * vpp + t;
    uint4* sp = staging + (ispos ? ((u64)__ldg(ispos + w) * G + g) : ((u64)w * sw + (u64)g * sg)) * vpp + t;
    const uint4* src = (MODE == MV_GATHER) ? pp : sp;
    uint4* dst = (MODE == MV_GATHER) ? sp : pp;
    u64 h = (u64)(t + 1) * C1, gq = (u64)(t + 1) * C4;
    for (u32 j0 = 0; j0 < vpt; j0 += UNR) {
      uint4 v[UNR];
#pragma unroll
      for (int jj = 0; jj < UNR; ++jj)
        if (j0 + jj < vpt) v[jj] = ld_stream(src + (u64)(j0 + jj) * LANES);
#pragma unroll
      for (int jj = 0; jj < UNR; ++jj)
        if (j0 + jj < vpt) {
          if (MODE != MV_DIGEST) st_stream(dst + (u64)(j0 + jj) * LANES, v[jj]);
          fold2(h, gq, v[jj]);
        }
    }
    const u64 s = warp_sum64(mixL(h)), s2 = warp_sum64(mixL(gq));
    if ((t & 31) == 0) { u64* o = part + ((u64)u * WPC + (t >> 5)) * 2; o[0] = s; o[1] = s2; }
  }
}

// ---------------------------------------------------------------------------------------------
// K2 / K4, TMA variant: the page is staged through shared memory with 1-D bulk copies
// (cp.async.bulk global->shared completing on an mbarrier; shared->global bulk store), so the
// LSU only sees conflict-free 16-byte shared loads for the checksum.  One elected thread issues
// the copies; a ring of STAGES tiles of TILE bytes keeps STAGES-1 loads in flight per CTA.
// Tiles of a page are consumed in order, so lane t still folds vectors t, t+256, ... in increasing
// order.  Persistent grid: CTA c handles pages c, c+grid, ...
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ u32 smem_u32(const void* p) { return (u32)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(u64* bar, u32 count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(u64* bar, u32 bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(u64* bar, u32 parity) {
  asm volatile(
      "{\n .reg .pred p;\n WAIT_%=:\n"
      " mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      " @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}\n" :: "r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, u32 bytes, u64* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               :: "r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* gdst, const void* smem_src, u32 bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
               :: "l"(gdst), "r"(smem_u32(smem_src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() {
  asm volatile("cp.async.bulk.wait_group.read %0;" :: "n"(N) : "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ void mbar_arrive(u64* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(smem_u32(bar)) : "memory");
}

// Warp roles: NG consumer groups of 8 warps (= the 256 checksum lanes of one page each; group g folds the CTA's pages
// g, g+NG, ...), then one load-producer warp and one store-issuer warp (lane 0 of each).  Every group owns a ring of
// STAGES tiles, so each mbarrier is waited on by the same warps in every phase.  full[s]: tile landed (tx bytes).
// empty[s]: the group's 8 warps (+ the store issuer once its bulk store has finished reading the stage) released the
// stage.  No block barrier in the steady state.  NG = 2 keeps four folding warps per scheduler: the mum fold (R22) is
// a chain of dependent IMAD.WIDEs, and two warps per scheduler could not hide its latency.
template <int NG> constexpr int tma_threads() { return NG * LANES + 64; }

template <int MODE, int STAGES, int TILE, int NG>
__global__ void __launch_bounds__(NG * LANES + 64, 1)
k_move_hash_tma(u8* __restrict__ pool, u8* __restrict__ staging, const u32* __restrict__ phys,
                u64* __restrict__ part, u32 n_items, u32 G, u32 NB, u32 page_bytes,
                const u32* __restrict__ iw, const u32* __restrict__ ispos, u32 sw, u32 sg) {
  extern __shared__ __align__(128) u8 smem[];
  __shared__ __align__(8) u64 full[NG * STAGES];
  __shared__ __align__(8) u64 empty[NG * STAGES];
  const u32 t = threadIdx.x, warp = t >> 5;
  constexpr u32 NCW = NG * WPC;                          // consumer warps
  const u32 n_pages = n_items * G;
  const u32 tpp = page_bytes / TILE;                     // tiles per page (page % TILE == 0)
  constexpr u32 VT = TILE / (16 * LANES);                // vectors per lane per tile
  if (t == 0) {
    for (int s = 0; s < NG * STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], WPC + (MODE != MV_DIGEST ? 1 : 0)); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  // this CTA's pages: blockIdx.x + k*grid, k = 0..my_pages-1; page k belongs to group k % NG and is that group's
  // (k / NG)-th page; its tile `tile` is the group's j-th tile, staged in ring slot j % STAGES in phase j / STAGES
  const u32 my_pages = (n_pages > blockIdx.x) ? (n_pages - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
  const u64 n_tiles = (u64)my_pages * tpp;
  auto slot = [&](u32 k, u32 tile, u32& s, u64& j) {
    j = (u64)(k / NG) * tpp + tile;
    s = (k % NG) * STAGES + (u32)(j % STAGES);
  };
  auto addr = [&](u32 k, u32 tile, u8*& gsrc, u8*& gdst, bool& skip) {
    const u32 u = blockIdx.x + k * gridDim.x;
    const u32 w = u / G, g = u - w * G;
    u32 b = 0;
    skip = false;
    if (MODE != MV_DIGEST) { b = __ldg(phys + (iw ? __ldg(iw + w) : w)); skip = (b == SKIP); if (skip) b = 0; }
    u8* pp = pool + ((u64)g * NB + b) * page_bytes + (u64)tile * TILE;
    u8* sp = staging + (ispos ? ((u64)__ldg(ispos + w) * G + g) : ((u64)w * sw + (u64)g * sg)) * page_bytes + (u64)tile * TILE;
    gsrc = (MODE == MV_GATHER) ? pp : sp;
    gdst = (MODE == MV_GATHER) ? sp : pp;
  };
  if (warp == NCW) {                                       // ---- load producer
    if (t == NCW * 32) {
      for (u64 q = 0; q < n_tiles; ++q) {
        const u32 k = (u32)(q / tpp), tile = (u32)(q - (u64)k * tpp);
        u32 s; u64 j; slot(k, tile, s, j);
        if (j >= STAGES) mbar_wait(&empty[s], (u32)(((j / STAGES) - 1) & 1));
        u8 *gs, *gd; bool skip; addr(k, tile, gs, gd, skip);
        mbar_expect_tx(&full[s], TILE);
        bulk_g2s(smem + s * TILE, gs, TILE, &full[s]);
      }
    }
  } else if (warp == NCW + 1) {                            // ---- store issuer
    if (MODE != MV_DIGEST && t == NCW * 32 + 32) {
      u32 prev = 0;
      for (u64 q = 0; q < n_tiles; ++q) {
        const u32 k = (u32)(q / tpp), tile = (u32)(q - (u64)k * tpp);
        u32 s; u64 j; slot(k, tile, s, j);
        mbar_wait(&full[s], (u32)((j / STAGES) & 1));
        u8 *gs, *gd; bool skip; addr(k, tile, gs, gd, skip);
        if (!skip) bulk_s2g(gd, smem + s * TILE, TILE);
        bulk_commit();
        if (q > 0) { bulk_wait_read<1>(); mbar_arrive(&empty[prev]); }   // the previous store drained its stage
        prev = s;
      }
      if (n_tiles) { bulk_wait_read<0>(); mbar_arrive(&empty[prev]); }
      asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    }
  } else {                                                 // ---- consumers: lane tl of group grp folds vectors tl, tl+256, ...
    const u32 grp = warp / WPC, tl = t - grp * LANES, wl = warp - grp * WPC;
    for (u32 k = grp; k < my_pages; k += NG) {
      u64 h = (u64)(tl + 1) * C1, gq = (u64)(tl + 1) * C4;
      for (u32 tile = 0; tile < tpp; ++tile) {
        u32 s; u64 j; slot(k, tile, s, j);
        mbar_wait(&full[s], (u32)((j / STAGES) & 1));
        const uint4* sv = reinterpret_cast<const uint4*>(smem + s * TILE) + tl;
#pragma unroll
        for (u32 v = 0; v < VT; ++v) fold2(h, gq, sv[v * LANES]);
        asm volatile("" :: "l"(h), "l"(gq) : "memory");    // the fold consumed the tile: its shared loads have completed
        __syncwarp();
        if ((t & 31) == 0) mbar_arrive(&empty[s]);         // this warp releases the stage
      }
      bool skip = false;
      const u32 u = blockIdx.x + k * gridDim.x;
      if (MODE != MV_DIGEST) { const u32 w = u / G; skip = __ldg(phys + (iw ? __ldg(iw + w) : w)) == SKIP; }
      const u64 sum = warp_sum64(mixL(h)), sum2 = warp_sum64(mixL(gq));
      if ((t & 31) == 0 && !skip) { u64* o = part + ((u64)u * WPC + wl) * 2; o[0] = sum; o[1] = sum2; }
    }
  }
}

// Per-block digests from the warp partial sums: page_digest(g) = (sum of its 8 partials, per family),
// d = mixF( sum_g mixL(p_g ^ (g+1)*C3) ),  e = mixF( sum_g mixL(q_g ^ (g+1)*C5) ).  One warp per work item.
__global__ void k_block_digest(const u64* __restrict__ part, const u32* __restrict__ phys, u64* __restrict__ d_out,
                               u64* __restrict__ e_out, u32 n_items, u32 G, const u32* __restrict__ iw) {
  const u32 w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (w >= n_items) return;
  const u32 wo = iw ? __ldg(iw + w) : w;            // output (and phys) position of item w
  if (phys && __ldg(phys + wo) == SKIP) { if (lane == 0) { d_out[wo] = 0; e_out[wo] = 0; } return; }
  u64 s = 0, t = 0;
  for (u32 g = lane; g < G; g += 32) {
    const u64* p = part + ((u64)w * G + g) * (WPC * 2);
    u64 pd = 0, qd = 0;
#pragma unroll
    for (int i = 0; i < WPC; ++i) { pd += p[2 * i]; qd += p[2 * i + 1]; }
    s += mixL(pd ^ ((u64)(g + 1) * C3));
    t += mixL(qd ^ ((u64)(g + 1) * C5));
  }
  s = warp_sum64(s); t = warp_sum64(t);
  if (lane == 0) { d_out[wo] = mixF(s); e_out[wo] = mixF(t); }
}

// ---------------------------------------------------------------------------------------------
// K1: predicate.  One warp per claim; lane l looks at table entries l, l+32, ...  Block i holds
// tokens [i*BS, min(P,(i+1)*BS)); it is complete iff fill[bt[i]] >= that count.  The leading run
// ends inside the first incomplete block: M = i0*BS + fill[bt[i0]], or P when all are complete.
// ---------------------------------------------------------------------------------------------
__global__ void k_pred(const Desc* __restrict__ desc, Res* __restrict__ res, u32 n, const u32* __restrict__ bt,
                       const u8* __restrict__ fill, u32 BS) {
  const u32 k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (k >= n) return;
  const Desc d = desc[k];
  if (!(d.flags & D_ELIG)) { if (lane == 0) res[k] = Res{0, 0, 0}; return; }
  u32 M = d.P;
  for (u32 base = 0; base < d.bt_len; base += 32) {
    const u32 i = base + lane;
    u32 f = 0; bool inc = false;
    if (i < d.bt_len) {
      f = fill[bt[d.bt_off + i]];
      const u32 rem = d.P - i * BS, cap = rem < BS ? rem : BS;
      inc = f < cap;
    }
    const u32 mask = __ballot_sync(0xFFFFFFFFu, inc);
    if (mask) {
      const int j = __ffs(mask) - 1;
      M = (base + j) * BS + __shfl_sync(0xFFFFFFFFu, f, j);
      break;
    }
  }
  if (lane == 0) res[k] = Res{M >= d.N ? (u32)R_OK : 0u, M, 0};
}

// block-wide inclusive scan of one u32 per thread (blockDim.x <= 1024)
__device__ __forceinline__ u32 block_scan_incl(u32 v, u32* warp_tot /*[32]*/, u32& total) {
  const u32 lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { u32 o = __shfl_up_sync(0xFFFFFFFFu, v, d); if (lane >= (u32)d) v += o; }
  __syncthreads();
  if (lane == 31) warp_tot[wid] = v;
  __syncthreads();
  if (wid == 0) {
    u32 x = lane < nw ? warp_tot[lane] : 0;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { u32 o = __shfl_up_sync(0xFFFFFFFFu, x, d); if (lane >= (u32)d) x += o; }
    warp_tot[lane] = x;
  }
  __syncthreads();
  total = warp_tot[nw - 1];
  return v + (wid ? warp_tot[wid - 1] : 0);
}

// K1: exclusive scan of nb over the eligible claims of a batch -> off[0..n].  One CTA.
__global__ void k_offsets(const Desc* __restrict__ desc, u32 n, u32* __restrict__ off) {
  __shared__ u32 wt[32];
  u32 carry = 0;
  for (u32 base = 0; base < n; base += blockDim.x) {
    const u32 k = base + threadIdx.x;
    const u32 c = (k < n && (desc[k].flags & D_ELIG)) ? desc[k].nb : 0;
    u32 tot;
    const u32 inc = block_scan_incl(c, wt, tot);
    if (k < n) off[k] = carry + inc - c;
    carry += tot;
    __syncthreads();
  }
  if (threadIdx.x == 0) off[n] = carry;
}

// K1: compaction.  Offload: phys[off_k+i] = bt[bt_off_k+i].  Restore: the allocation list is the
// work list; write it into the claim's new table and mark suppressed transfers.
__global__ void k_worklist(const Desc* __restrict__ desc, const Res* __restrict__ res, u32 n,
                           const u32* __restrict__ off, u32* __restrict__ bt, const u32* __restrict__ alloc,
                           u32* __restrict__ phys, int restore) {
  const u32 k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (k >= n) return;
  const Desc d = desc[k];
  if (!restore) {
    if (!(d.flags & D_ELIG)) return;
    for (u32 i = lane; i < d.nb; i += 32) phys[off[k] + i] = bt[d.bt_off + i];
  } else {
    if (!(res[k].flag & R_SERVED)) return;
    for (u32 i = lane; i < d.nb; i += 32) {
      const u32 b = alloc[off[k] + i];
      bt[d.bt_off + i] = b;
      phys[off[k] + i] = (d.flags & D_XFER) ? SKIP : b;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// K3: chain.  H = seed(C); H = H*A + d_i.  The step is the affine map x -> x*A + d_i; maps
// compose associatively as (a1,b1)*(a2,b2) = (a1*a2, b1*a2 + b2), so an inclusive warp scan of 32
// blocks gives the tile's map and H advances one tile per iteration.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ u64 chain_tile(u64 h, u64 d, bool valid) {
  const u32 lane = threadIdx.x & 31;
  u64 a = valid ? CA : 1ull, b = valid ? d : 0ull;
#pragma unroll
  for (int s = 1; s < 32; s <<= 1) {
    const u64 pa = shfl_up64(a, s), pb = shfl_up64(b, s);
    if (lane >= (u32)s) { b = pb * a + b; a = pa * a; }
  }
  a = __shfl_sync(0xFFFFFFFFu, a, 31);
  b = __shfl_sync(0xFFFFFFFFu, b, 31);
  return h * a + b;
}

__global__ void k_chain(const Desc* __restrict__ desc, Res* __restrict__ res, u32 n, const u32* __restrict__ off,
                        const u64* __restrict__ d_tmp, const u64* __restrict__ e_tmp, u64* __restrict__ dg,
                        u64* __restrict__ dg2) {
  const u32 k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (k >= n) return;
  const Desc d = desc[k];
  if (!(d.flags & D_ELIG)) { if (lane == 0) res[k] = Res{0, 0, 0}; return; }
  u64 h = mixF(d.id ^ C3);
  for (u32 base = 0; base < d.nb; base += 32) {
    const u32 i = base + lane;
    const bool valid = i < d.nb;
    const u64 x = valid ? d_tmp[off[k] + i] : 0;
    if (valid) { dg[d.dg_off + i] = x; dg2[d.dg_off + i] = e_tmp[off[k] + i]; }
    h = chain_tile(h, x, valid);
  }
  if (lane == 0) res[k] = Res{R_OK | R_SERVED, d.nb, h};
}

// ---------------------------------------------------------------------------------------------
// K5: restore plan.  One CTA.  (1) free count at entry; (2) inclusive scan of nb over eligible
// claims in batch order: claim k is served iff the running sum <= free count (nb >= 1, so the
// served set is a prefix of the eligible claims); (3) the r-th free block in ascending id order,
// r < total, goes to alloc[r].  Work-list offsets off[] are the same scan.
// ---------------------------------------------------------------------------------------------
__global__ void k_restore_plan(const Desc* __restrict__ desc, Res* __restrict__ res, u32 n, u32* __restrict__ off,
                               u8* __restrict__ used, u32* __restrict__ ref, u32 NB, u32* __restrict__ alloc,
                               u32* __restrict__ counters /*[2]: nfree, total*/) {
  __shared__ u32 wt[32];
  __shared__ u32 s_nfree, s_total;
  u32 cnt = 0;
  for (u32 b = threadIdx.x; b < NB; b += blockDim.x) cnt += used[b] == 0;
  { u32 tot; block_scan_incl(cnt, wt, tot); if (threadIdx.x == 0) { s_nfree = tot; s_total = 0; } }
  __syncthreads();
  const u32 nfree = s_nfree;
  u32 carry = 0;
  for (u32 base = 0; base < n; base += blockDim.x) {
    const u32 k = base + threadIdx.x;
    const bool el = k < n && (desc[k].flags & D_ELIG);
    const u32 c = el ? desc[k].nb : 0;
    u32 tot;
    const u32 inc = carry + block_scan_incl(c, wt, tot);
    if (k < n) {
      const bool served = el && inc <= nfree;
      res[k] = Res{served ? (u32)R_SERVED : 0u, 0, 0};
      off[k] = served ? inc - c : 0xFFFFFFFFu;
      if (served) atomicMax(&s_total, inc);
    }
    carry += tot;
    __syncthreads();
  }
  __syncthreads();
  const u32 total = s_total;
  if (threadIdx.x == 0) { off[n] = total; counters[0] = nfree; counters[1] = total; }
  for (u32 k = threadIdx.x; k < n; k += blockDim.x) if (off[k] == 0xFFFFFFFFu) off[k] = total;
  carry = 0;
  for (u32 base = 0; base < NB && carry < total; base += blockDim.x) {
    const u32 b = base + threadIdx.x;
    const u32 f = (b < NB && used[b] == 0) ? 1u : 0u;
    u32 tot;
    const u32 r = carry + block_scan_incl(f, wt, tot) - f;
    if (f && r < total) { alloc[r] = b; used[b] = 1; ref[b] = 1; }
    carry += tot;
    __syncthreads();
  }
}

// ok: fill of the claim's new blocks := leading tokens they hold.  not ok: the new blocks are freed.  (one warp)
__device__ __forceinline__ void apply_verdict(const Desc& d, bool ok, const u32* __restrict__ bt, u8* __restrict__ used,
                                              u32* __restrict__ ref, u8* __restrict__ fill, u32 BS) {
  const u32 lane = threadIdx.x & 31;
  for (u32 i = lane; i < d.nb; i += 32) {
    const u32 b = bt[d.bt_off + i];
    if (ok) { const u32 rem = d.M - i * BS; fill[b] = (u8)(rem < BS ? rem : BS); }
    else { used[b] = 0; ref[b] = 0; fill[b] = 0; }
  }
}

// K4 tail: verdict per served claim.  bad = first block whose recomputed digest differs; ok iff the
// transfer was not suppressed, no block differs and the recomputed chain equals the recorded one.
// ok: fill of the new blocks := leading tokens they hold.  not ok: the new blocks are freed.
__global__ void k_verify(const Desc* __restrict__ desc, Res* __restrict__ res, u32 n, const u32* __restrict__ off,
                         const u64* __restrict__ d_tmp, const u64* __restrict__ e_tmp, const u64* __restrict__ dg,
                         const u64* __restrict__ dg2, const u32* __restrict__ bt,
                         u8* __restrict__ used, u32* __restrict__ ref, u8* __restrict__ fill, u32 BS, int apply) {
  const u32 k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (k >= n) return;
  if (!(res[k].flag & R_SERVED)) return;
  const Desc d = desc[k];
  u32 bad = 0xFFFFFFFFu;
  bool ok = !(d.flags & D_XFER);
  if (ok) {
    u64 h = mixF(d.id ^ C3);
    for (u32 base = 0; base < d.nb; base += 32) {
      const u32 i = base + lane;
      const bool valid = i < d.nb;
      const u64 x = valid ? d_tmp[off[k] + i] : 0;
      const u32 mm = __ballot_sync(0xFFFFFFFFu, valid && (x != dg[d.dg_off + i] || e_tmp[off[k] + i] != dg2[d.dg_off + i]));
      if (mm && bad == 0xFFFFFFFFu) bad = base + __ffs(mm) - 1;
      h = chain_tile(h, x, valid);
    }
    ok = bad == 0xFFFFFFFFu && h == d.chain;
  }
  if (apply) apply_verdict(d, ok, bt, used, ref, fill, BS);          // TP mode applies the MERGED verdict later (k_tp_apply)
  if (lane == 0) res[k] = Res{R_SERVED | (ok ? (u32)R_OK : 0u), bad, d.chain};
}

// ---------------------------------------------------------------------------------------------
// NEXT-4: TP-sharded KV, one common verdict (DESIGN.md 8 / R24).  Every rank verifies its kv_head shard
// (k_verify, apply = 0) and publishes one 8-byte record per claim: flags (1 served, 2 locally ok) and bad.  k_tp_push
// stores this rank's records straight into every peer's mailbox (peer-mapped device memory: the stores cross NVLink)
// and then releases a per-source epoch flag; k_tp_merge folds the G records of each claim -- ok = AND, bad = min over
// the failing ranks -- into res[], from a gathered buffer (all-gather path) or from this rank's own mailbox; k_tp_apply
// is the second half of k_verify under the merged verdict.  No kernel ever waits for another rank: a mailbox whose
// flags are not at the expected epoch is reported (k_tp_ready) and the host refuses the commit.
// ---------------------------------------------------------------------------------------------
struct TpVerdict { u32 flags, bad; };
enum { TV_SERVED = 1, TV_OK = 2 };
constexpr int TP_MAX_RANKS = 16;
struct TpPeers { u64* flag[TP_MAX_RANKS]; TpVerdict* rec[TP_MAX_RANKS]; };   // per peer: its epoch flags, its record area

__global__ void k_tp_verdicts(const Res* __restrict__ res, u32 n, TpVerdict* __restrict__ out) {
  const u32 k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const Res r = res[k];
  out[k] = (r.flag & R_SERVED) ? TpVerdict{(u32)TV_SERVED | ((r.flag & R_OK) ? (u32)TV_OK : 0u), r.val} : TpVerdict{0u, 0xFFFFFFFFu};
}
// one CTA: records to every open peer (slot [my_rank][k] of the peer's area), then the epoch flags, released system-wide
__global__ void k_tp_push(const TpVerdict* __restrict__ local, u32 n, TpPeers peers, u32 G, u32 my_rank, u32 stride, u64 epoch) {
  for (u32 p = 0; p < G; ++p) {
    if (!peers.rec[p]) continue;
    TpVerdict* dst = peers.rec[p] + (u64)my_rank * stride;
    for (u32 k = threadIdx.x; k < n; k += blockDim.x) dst[k] = local[k];
  }
  __threadfence_system();
  __syncthreads();
  if (threadIdx.x < G && peers.flag[threadIdx.x]) {
    asm volatile("st.release.sys.global.u64 [%0], %1;" :: "l"(peers.flag[threadIdx.x] + my_rank), "l"(epoch) : "memory");
  }
}
__global__ void k_tp_ready(const u64* __restrict__ flags, u32 G, u64 epoch, u32* __restrict__ not_ready) {
  if (threadIdx.x < G) {
    u64 v;
    asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(flags + threadIdx.x) : "memory");
    if (v != epoch) atomicAdd(not_ready, 1u);
  }
}
// src[r*stride + k] = record of rank r for batch entry k.  A rank that disagrees on `served` is a call-level error.
__global__ void k_tp_merge(Res* __restrict__ res, u32 n, const TpVerdict* __restrict__ src, u32 stride, u32 G,
                           u32* __restrict__ errors) {
  const u32 k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  Res r = res[k];
  const u32 served = (r.flag & R_SERVED) ? (u32)TV_SERVED : 0u;
  bool ok = true; u32 bad = 0xFFFFFFFFu;
  for (u32 q = 0; q < G; ++q) {
    const TpVerdict v = src[(u64)q * stride + k];
    if ((v.flags & TV_SERVED) != served) { atomicAdd(errors, 1u); return; }
    if (!(v.flags & TV_OK)) { ok = false; bad = v.bad < bad ? v.bad : bad; }
  }
  if (!served) return;
  r.flag = R_SERVED | (ok ? (u32)R_OK : 0u);
  r.val = ok ? 0xFFFFFFFFu : bad;
  res[k] = r;
}
__global__ void k_tp_apply(const Desc* __restrict__ desc, const Res* __restrict__ res, u32 n, const u32* __restrict__ bt,
                           u8* __restrict__ used, u32* __restrict__ ref, u8* __restrict__ fill, u32 BS) {
  const u32 k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (k >= n) return;
  const Res r = res[k];
  if (!(r.flag & R_SERVED)) return;
  apply_verdict(desc[k], (r.flag & R_OK) != 0, bt, used, ref, fill, BS);
}

// K5: drop the claim's references to all its table blocks; a block whose count reaches 0 is free.
__global__ void k_unref(const Desc* __restrict__ desc, u32 n, const u32* __restrict__ bt, u8* __restrict__ used,
                        u32* __restrict__ ref) {
  const u32 k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (k >= n) return;
  const Desc d = desc[k];
  if (!(d.flags & D_ELIG)) return;
  for (u32 i = lane; i < d.bt_len; i += 32) {
    const u32 b = bt[d.bt_off + i];
    const u32 old = atomicSub(&ref[b], 1u);
    if (old == 1u) used[b] = 0;
  }
}

__global__ void k_mark(const u32* __restrict__ ids, u32 n, u8* __restrict__ used, const u32* __restrict__ ref, int val) {
  const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const u32 b = ids[i];
  if (val) used[b] = 1; else if (ref[b] == 0) used[b] = 0;
}

// a0: table validation.  One CTA per candidate at a time; `bm` is this CTA's private NB-bit map
// (all zero between candidates).  Valid iff every id is in range, used, and distinct.
__global__ void k_accept(const Desc* __restrict__ desc, Res* __restrict__ res, u32 n, const u32* __restrict__ up,
                         u32* __restrict__ bt, const u8* __restrict__ used, u32* __restrict__ ref, u32 NB,
                         u32* __restrict__ bitmaps) {
  u32* bm = bitmaps + (size_t)blockIdx.x * ((NB + 31) / 32);
  for (u32 k = blockIdx.x; k < n; k += gridDim.x) {
    const Desc d = desc[k];
    if (!(d.flags & D_ELIG)) { if (threadIdx.x == 0) res[k] = Res{0, 0, 0}; continue; }
    int bad = 0;
    for (u32 i = threadIdx.x; i < d.bt_len; i += blockDim.x) {
      const u32 b = up[d.src_off + i];
      if (b >= NB || !used[b]) { bad = 1; continue; }
      const u32 bit = 1u << (b & 31);
      if (atomicOr(&bm[b >> 5], bit) & bit) bad = 1;
    }
    bad = __syncthreads_or(bad);
    for (u32 i = threadIdx.x; i < d.bt_len; i += blockDim.x) {
      const u32 b = up[d.src_off + i];
      if (b < NB) bm[b >> 5] = 0;
      if (!bad) { bt[d.bt_off + i] = b; atomicAdd(&ref[b], 1u); }
    }
    if (threadIdx.x == 0) res[k] = Res{bad ? 0u : (u32)R_OK, 0, 0};
    __syncthreads();
  }
}

// ---------------------------------------------------------------------------------------------
// K6: outcome emission.  One CTA.  Per claim of the batch, in batch order, the number of records
// follows from the call and the claim's result; an exclusive scan assigns record offsets, so all
// records of claim k precede those of claim k+1 and seq is gap-free (P:L27 order per claim).
// ---------------------------------------------------------------------------------------------
__global__ void k_emit(const Desc* __restrict__ desc, const Res* __restrict__ res, u32 n, int mode,
                       Event* __restrict__ ring, u32 ring_cap, u64* __restrict__ ev_count, u64 request_id, int tp) {
  __shared__ u32 wt[32];
  const u64 seq0 = *ev_count;
  u32 carry = 0, carry_b = 0;
  // what a failed restoration means for claim k: refusal (per claim, or deferred to the request's run), demotion, expiry
  auto blocks_request = [&](const Desc& d, const Res& r) {
    return mode == EM_RESTORE && request_id != 0 && (r.flag & R_SERVED) && !(r.flag & R_OK) && d.pad == POL_REFUSE;
  };
  for (u32 base = 0; base < n; base += blockDim.x) {
    const u32 k = base + threadIdx.x;
    Desc d; Res r; u32 c = 0;
    if (k < n) {
      d = desc[k]; r = res[k];
      if (mode == EM_RESTORE) c = (r.flag & R_SERVED) ? ((r.flag & R_OK) ? 2u : (blocks_request(d, r) ? 3u : 4u)) : 0u;
      else if (mode == EM_DEMOTE || mode == EM_CONFLICT) c = (d.flags & D_ELIG) ? 1u : 0u;
      else c = (r.flag & R_OK) ? 1u : 0u;
    }
    u32 tot;
    const u32 o = carry + block_scan_incl(c, wt, tot) - c;
    if (c) {
      u64 s = seq0 + o;
      auto put = [&](u32 code, u32 aux, u64 arg) {
        ring[s % ring_cap] = Event{s, d.id, code, aux, arg};
        ++s;
      };
      if (mode == EM_ACCEPT) put(EV_ACCEPTED, d.N, d.P);
      else if (mode == EM_MATERIALIZE) put(EV_MATERIALIZED, r.val, 0);
      else if (mode == EM_OFFLOAD) put(EV_OFFLOADED, d.nb, tp ? 0 : r.chain);   // TP: chains are rank-local, streams identical
      else if (mode == EM_DEMOTE) put(EV_DEMOTED, d.bt_len, request_id);          // victim: the boundary precedes the loss
      else if (mode == EM_CONFLICT) put(EV_CONFLICT_REFUSED, REQ_FLAG | n, request_id);   // all n descs are blocking claims
      else {
        put(EV_RESTORE_REQUIRED, d.M, 0);
        if (r.flag & R_OK) put(EV_RESTORED, d.nb, tp ? 0 : d.chain);
        else {
          put(EV_LOAD_FAILED, r.val, 0);
          put(EV_RESTORATION_FAILED, 0, 0);
          if (d.pad == POL_DEMOTE) put(EV_DEMOTED, 0, 0);
          else if (d.pad == POL_EXPIRE) put(EV_EXPIRED, 0, 0);
          else if (request_id == 0) put(EV_ACTIVE_REQUEST_REFUSED, 1, d.id);
        }
      }
    }
    carry += tot;
    __syncthreads();
  }
  __syncthreads();
  if (mode == EM_RESTORE && request_id != 0) {
    // request-level refusal: one record per blocking claim, batch order, after the per-claim records;
    // aux = REQ_FLAG | size of the failed subset, arg = request id (blocking_claim_ids = the run's claim ids)
    u32 K = 0;
    for (u32 base = 0; base < n; base += blockDim.x) {
      const u32 k = base + threadIdx.x;
      const u32 b = (k < n && blocks_request(desc[k], res[k])) ? 1u : 0u;
      u32 tot;
      block_scan_incl(b, wt, tot);
      K += tot;
      __syncthreads();
    }
    for (u32 base = 0; base < n; base += blockDim.x) {
      const u32 k = base + threadIdx.x;
      const u32 b = (k < n && blocks_request(desc[k], res[k])) ? 1u : 0u;
      u32 tot;
      const u32 o = carry_b + block_scan_incl(b, wt, tot) - b;
      if (b) {
        const u64 s = seq0 + carry + o;
        ring[s % ring_cap] = Event{s, desc[k].id, EV_ACTIVE_REQUEST_REFUSED, REQ_FLAG | K, request_id};
      }
      carry_b += tot;
      __syncthreads();
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) *ev_count = seq0 + carry + carry_b;
}

// ---------------------------------------------------------------------------------------------
// K5, allocator-side protection (NEXT-3; P:L85 victim_exclusion_before_violation, P:L270 allocator_hook).
// Candidates arrive in victim order (unprotected first, then protected; acceptance order inside each group).
// Evicting the first m candidates frees the blocks whose every holder is among them: block b is freed by the
// LAST of its holders in list order, so gain[k] = #{b in table k : posmax[b] == k+1} with posmax[b] = the largest
// list position (+1) of a holder of b, and the free count after evicting m claims is F + sum_{k<m} gain[k].
// ---------------------------------------------------------------------------------------------
__global__ void k_vic_posmax(const Desc* __restrict__ desc, u32 n, const u32* __restrict__ bt, u32* __restrict__ posmax) {
  const u32 k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (k >= n) return;
  const Desc d = desc[k];
  for (u32 i = lane; i < d.bt_len; i += 32) atomicMax(&posmax[bt[d.bt_off + i]], k + 1);
}
__global__ void k_vic_gain(const Desc* __restrict__ desc, u32 n, const u32* __restrict__ bt, const u32* __restrict__ posmax,
                           u32* __restrict__ gain) {
  const u32 k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (k >= n) return;
  const Desc d = desc[k];
  u32 g = 0;
  for (u32 i = lane; i < d.bt_len; i += 32) g += posmax[bt[d.bt_off + i]] == k + 1;
  g = warp_sum32(g);
  if (lane == 0) gain[k] = g;
}
// One CTA.  F = free blocks; m = the shortest prefix with F + sum gain >= need.  U = number of unprotected candidates.
// out[0] = outcome (VO_*), out[1] = first list position concerned, out[2] = one past the last, out[3] = F.
__global__ void k_vic_decide(const u32* __restrict__ gain, u32 n, u32 U, u32 need, const u8* __restrict__ used, u32 NB,
                             u32* __restrict__ out) {
  __shared__ u32 wt[32];
  __shared__ u32 s_m;
  u32 cnt = 0;
  for (u32 b = threadIdx.x; b < NB; b += blockDim.x) cnt += used[b] == 0;
  u32 F;
  block_scan_incl(cnt, wt, F);
  if (threadIdx.x == 0) s_m = 0xFFFFFFFFu;
  __syncthreads();
  u32 carry = F;
  for (u32 base = 0; base < n && F < need; base += blockDim.x) {
    const u32 k = base + threadIdx.x;
    u32 tot;
    const u32 inc = carry + block_scan_incl(k < n ? gain[k] : 0u, wt, tot);
    if (k < n && inc >= need) atomicMin(&s_m, k + 1);
    carry += tot;
    __syncthreads();
    if (s_m != 0xFFFFFFFFu) break;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    const u32 m = s_m;
    u32 oc, lo = 0, hi = 0;
    if (F >= need) oc = VO_FITS;
    else if (m != 0xFFFFFFFFu && m <= U) { oc = VO_EVICT; lo = 0; hi = m; }
    else if (U == n) oc = VO_NOFREE;
    else { oc = VO_CONFLICT; lo = U; hi = m != 0xFFFFFFFFu ? m : n; }
    out[0] = oc; out[1] = lo; out[2] = hi; out[3] = F;
  }
}
// the protected resident footprint as a byte map (rc_protected_map)
__global__ void k_prot_map(const Desc* __restrict__ desc, u32 n, const u32* __restrict__ bt, u8* __restrict__ map) {
  const u32 k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (k >= n) return;
  const Desc d = desc[k];
  if (!(d.flags & D_PROT)) return;
  for (u32 i = lane; i < d.bt_len; i += 32) map[bt[d.bt_off + i]] = 1;
}

// Small metadata transfers (descriptors, tables, results, event records: bytes to a few MB) between mapped pinned host
// memory and device memory, word by word over PCIe.  The copy engines are left to the GiB-sized chunk copies: a 20 KB
// cudaMemcpyAsync queued behind one of those in an engine's FIFO waits tens of milliseconds.
__global__ void k_copy_words(u32* __restrict__ dst, const u32* __restrict__ src, u64 n_words) {
  for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n_words; i += (u64)gridDim.x * blockDim.x) dst[i] = src[i];
}

// Checked mode (RC_CHECK=1; compute-sanitizer is closed on this pool): every address a mover forms derives from its work
// items -- phys[w] (pool block), iw[w] (work position), ispos[w] (staged block) -- and the loop bounds, so validating the
// items before each launch bounds every access of that launch.  A violation sets the mapped flag; the host refuses to
// complete the operation.
__global__ void k_check_items(const u32* __restrict__ phys, u32 n_items, u32 NB, const u32* __restrict__ iw, u32 iw_limit,
                              const u32* __restrict__ ispos, u32 ispos_limit, u32* __restrict__ flag) {
  const u32 w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= n_items) return;
  bool bad = false;
  u32 pw = w;
  if (iw) { pw = iw[w]; bad |= pw >= iw_limit; }
  if (phys && !bad) { const u32 b = phys[pw]; bad |= (b >= NB && b != SKIP); }
  if (ispos) bad |= ispos[w] >= ispos_limit;
  if (bad) *flag = 1u;
}

// rc_set_fill: fill[ids[i]] = vals[i] (the caller's materialization marks, sent as host arrays)
__global__ void k_fill_write(const u32* __restrict__ ids, const u8* __restrict__ vals, u32 n, u8* __restrict__ fill) {
  const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) fill[ids[i]] = vals[i];
}

// fault injection (CPU->GPU transfers only): flip bit 0 of the listed staged bytes
__global__ void k_bitflip(u8* staging, const u64* __restrict__ offs, u32 n) {
  const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) staging[offs[i]] ^= 0x01;
}

}  // namespace rck
