// rc_dedup.inl -- NEXT-2: content-addressed host store.  Included by librc.cu.
//
// Blocks are keyed by the 128-bit pair (d, e) of their two digests (both computed by the fused gather anyway).  Offload: every block is
// gathered and digested at HBM speed as before; per staging chunk the digests come back to the host (8 B per
// block), and only blocks whose key is not in the store are copied over the link.  Restore: the distinct
// blocks of the call are staged once (first appearance order) and the scatter kernel reads them through an
// item -> staged-block indirection, so a shared block crosses the link once per call; a claim with an injected
// BITFLIP gets private staged copies, which keeps the corruption -- and the attribution -- on that claim alone
// (P:L384).  Host space is granted as if every block were new (prefix sum, R7) and charged by content.
// The store is looked up and extended by rc_offload_begin (the keys come back chunk by chunk while the call runs); a
// restore's references to the store end when rc_wait(1) completes it.

static bool dedup_alloc_slot(rc_ctx* c, u32& slot, int& err) {
  u64 o;
  err = RC_OK;
  if (!c->host_alloc.alloc(1, o)) return false;
  slot = (u32)o;
  return true;
}

static void dedup_drop(rc_ctx* c, Claim& cl) {                  // the claim's references to the store
  for (size_t i = 0; i < cl.hkeys.size(); ++i) {
    auto it = c->store.find(cl.hkeys[i]);
    if (it == c->store.end()) continue;
    if (--it->second.second == 0) {
      c->host_alloc.release(it->second.first, 1);
      c->store.erase(it);
      c->host_used -= c->blk;
    }
  }
  cl.hkeys.clear(); cl.hslots.clear();
}

static int offload_begin_dedup(rc_ctx* c, uint32_t n, const uint64_t* id, int32_t* st) {
  if (c->off_open) return RC_ERR_BUSY;                     // one open offload: the keys come back through one host buffer
  const int slot_o = 0, oi = off_oi(slot_o), set = off_set(slot_o);
  Op& op = c->ops[oi];
  if (n == 0) return RC_OK;
  if (!id || !st || n > c->desc_cap) return RC_ERR_INVALID;
  if (!ev_room(c, n)) return RC_ERR_CAPACITY;
  Desc* hd = c->h_desc[set];
  op.cl.assign(n, nullptr);
  std::vector<u32> served;
  std::vector<u64> first_w;
  bool full = false;
  u64 T = 0, worst = c->host_used;
  std::vector<std::pair<u32, u32>> old_dg;
  auto rollback = [&]() {                                  // a negative return changes no claim (rc.h)
    for (size_t j = 0; j < served.size(); ++j) {
      Claim& cl = *op.cl[served[j]];
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
    if (cl.busy || (cl.state != RC_CS_MATERIALIZED && cl.state != RC_CS_RESIDENT_AGAIN)) { st[k] = RC_ST_BAD_STATE; continue; }
    if (full || worst + (u64)cl.nb * c->blk > c->cfg.host_store_bytes) { full = true; st[k] = RC_ST_NO_HOST_SPACE; continue; }
    worst += (u64)cl.nb * c->blk;
    u64 dgo;
    if (T + cl.nb > c->cap_entries || !c->dg_alloc.alloc(cl.nb, dgo)) { rollback(); return RC_ERR_CAPACITY; }
    old_dg.push_back({cl.dg_off, cl.dg_len});
    cl.dg_off = (u32)dgo; cl.dg_len = cl.nb;
    cl.hslots.clear(); cl.hkeys.clear();
    cl.busy = true;
    op.cl[k] = &cl;
    served.push_back(k);
    first_w.push_back(T);
    hd[k].P = cl.P; hd[k].N = cl.N; hd[k].M = cl.M; hd[k].nb = cl.nb; hd[k].bt_off = cl.bt_off; hd[k].bt_len = cl.bt_len;
    hd[k].dg_off = cl.dg_off; hd[k].flags = D_ELIG;
    T += cl.nb;
    st[k] = -1;
  }
  if (served.empty()) return RC_OK;
  for (auto& od : old_dg) if (od.second) c->dg_alloc.release(od.first, od.second);
  op.n = n; op.status = st; op.blocks = T; op.copy_bytes = 0; op.launches = 0;
  int rc;
  CK(to_dev(c, c->gather, c->d_desc[set], c->h_desc[set], (u64)n * sizeof(Desc)));
  k_offsets<<<1, 1024, 0, c->gather>>>(c->d_desc[set], n, c->d_off[set]);
  CKL();
  k_worklist<<<warps_grid(n), 256, 0, c->gather>>>(c->d_desc[set], c->d_res[set], n, c->d_off[set], c->d_bt, nullptr, c->d_phys[oi], 0);
  CKL();
  c->st.kernel_launches += 2;
  size_t ci_claim = 0;                                     // served claim that owns the current work position
  for (u64 w0 = 0; w0 < T; w0 += c->chunk_blocks) {
    const u64 w1 = std::min(T, w0 + c->chunk_blocks);
    const u32 slot = (u32)(c->chunk_seq[0]++ % c->R), m = (u32)(w1 - w0);
    if (c->slot_used[0][slot]) CK(cudaStreamWaitEvent(c->gather, c->ev_free[0][slot], 0));
    cudaEvent_t t0 = get_event(c), t1 = get_event(c);
    CK(cudaEventRecord(t0, c->gather));
    launch_move<MV_GATHER>(c, c->gather, c->staging[0][slot], c->d_phys[oi] + w0, c->part[0][slot], m);
    CKL();
    CK(cudaEventRecord(t1, c->gather));
    op.t_kernel.push_back({t0, t1});
    op.launches++;
    k_block_digest<<<warps_grid(m), 256, 0, c->gather>>>(c->part[0][slot], nullptr, c->d_dtmp[oi] + w0, c->d_etmp[oi] + w0, m, c->G, nullptr);
    CKL();
    c->st.kernel_launches++;
    CK(to_host(c, c->gather, c->h_dig + w0, c->d_dtmp[oi] + w0, (u64)m * 8));
    CK(to_host(c, c->gather, c->h_dig2 + w0, c->d_etmp[oi] + w0, (u64)m * 8));
    CK(cudaEventRecord(c->ev_ready[0][slot], c->gather));
    CK(cudaStreamSynchronize(c->gather));                  // the keys decide which blocks cross the link
    CK(cudaStreamWaitEvent(c->d2h, c->ev_ready[0][slot], 0));
    cudaEvent_t c0 = get_event(c), c1 = get_event(c);
    CK(cudaEventRecord(c0, c->d2h));
    u8 *ha = nullptr, *da = nullptr; u64 len = 0;
    for (u64 w = w0; w < w1; ++w) {
      while (ci_claim + 1 < served.size() && first_w[ci_claim + 1] <= w) ++ci_claim;
      Claim& cl = *op.cl[served[ci_claim]];
      const Key key(c->h_dig[w], c->h_dig2[w]);
      auto it = c->store.find(key);
      u32 hs;
      if (it != c->store.end()) { it->second.second++; hs = it->second.first; }
      else {
        if (!dedup_alloc_slot(c, hs, rc)) {               // cannot happen: space was granted by count at the top
          if (!rc) { c->poisoned = true; c->cuda_err = "internal: dedup host-store accounting"; rc = RC_ERR_CUDA; }
          return rc;                                       // sticky, like every error past the first enqueued copy
        }
        c->store.emplace(key, std::make_pair(hs, 1u));
        c->host_used += c->blk;
        u8* h = c->h_store + (u64)hs * c->blk;
        u8* d = c->staging[0][slot] + (w - w0) * c->blk;
        if (len && h == ha + len && d == da + len) len += c->blk;
        else {
          if (len) { CK(cudaMemcpyAsync(ha, da, len, cudaMemcpyDeviceToHost, c->d2h)); op.copy_bytes += len; }
          ha = h; da = d; len = c->blk;
        }
      }
      cl.hslots.push_back(hs); cl.hkeys.push_back(key);
    }
    if (len) { CK(cudaMemcpyAsync(ha, da, len, cudaMemcpyDeviceToHost, c->d2h)); op.copy_bytes += len; }
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

static int restore_begin_dedup(rc_ctx* c, uint32_t n, const uint64_t* id, int32_t* st) {
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
  CK(cudaStreamSynchronize(c->meta));
  // staged blocks in first-appearance order; items = (work position, staged block)
  std::vector<u32> su;                                     // staged index -> host slot
  std::vector<std::pair<u32, u32>> items;                  // (staged index, work position)
  std::vector<std::pair<u64, u64>> flips;                  // (staged index, byte in block)
  std::unordered_map<u32, u32> staged_of;                  // host slot -> staged index (this call)
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
    rc_fault flt{0, 0, 0};
    for (size_t f = 0; f < c->faults.size(); ++f)
      if (c->faults[f].claim_id == id[k]) { flt = c->faults[f]; c->faults.erase(c->faults.begin() + f); break; }
    if (flt.kind == RC_FAULT_XFER_ERROR) { hd[k].flags |= D_XFER; reupload = true; }
    else if (flt.kind == RC_FAULT_BITFLIP) {               // private staged copies: the corruption stays on this claim
      const u64 pos = flt.param % ((u64)cl.nb * c->blk);
      flips.push_back({su.size() + pos / c->blk, pos % c->blk});
      for (u32 i = 0; i < cl.nb; ++i) { items.push_back({(u32)su.size(), (u32)(T + i)}); su.push_back(cl.hslots[i]); }
    } else {
      for (u32 i = 0; i < cl.nb; ++i) {
        auto ins = staged_of.emplace(cl.hslots[i], (u32)su.size());
        if (ins.second) su.push_back(cl.hslots[i]);
        items.push_back({ins.first->second, (u32)(T + i)});
      }
    }
    T += cl.nb;
  }
  if (n_served == 0) return RC_OK;
  if (c->fault_flags & RC_FAULT_ALLOW_UNCLAIMED)
    for (size_t f = 0; f < c->faults.size();)
      if (c->faults[f].claim_id == 0) { c->st.generic_failures++; c->faults.erase(c->faults.begin() + f); } else ++f;
  op.n = n; op.status = st; op.blocks = items.size(); op.copy_bytes = 0; op.launches = 0;
  if (reupload && (rc = upload_desc(c, 1, n))) return rc;
  k_worklist<<<warps_grid(n), 256, 0, c->meta>>>(c->d_desc[1], c->d_res[1], n, c->d_off[1], c->d_bt, c->d_alloc, c->d_phys[1], 1);
  CKL();
  c->st.kernel_launches++;
  // group the items by staging chunk (staged index / chunk_blocks); upload (work position, staged block in chunk)
  std::stable_sort(items.begin(), items.end(), [&](const std::pair<u32, u32>& a, const std::pair<u32, u32>& b) {
    return a.first / c->chunk_blocks < b.first / c->chunk_blocks; });
  for (size_t j = 0; j < items.size(); ++j) { c->h_iw[j] = items[j].second; c->h_ispos[j] = (u32)(items[j].first % c->chunk_blocks); }
  if (!items.empty()) {
    CK(to_dev(c, c->meta, c->d_iw, c->h_iw, items.size() * 4));
    CK(to_dev(c, c->meta, c->d_ispos, c->h_ispos, items.size() * 4));
  }
  CK(cudaEventRecord(c->ev_plan[1], c->meta));
  CK(cudaStreamWaitEvent(c->scatter, c->ev_plan[1], 0));
  std::sort(flips.begin(), flips.end());
  size_t fi = 0, ji = 0;
  u64 flip_base = 0;
  u32 ci = 0;
  const u64 U = su.size();
  for (u64 u0 = 0; u0 < U; u0 += c->chunk_blocks, ++ci) {
    const u64 u1 = std::min(U, u0 + c->chunk_blocks);
    const u32 slot = (u32)(c->chunk_seq[1]++ % c->R);
    if (c->slot_used[1][slot]) CK(cudaStreamWaitEvent(c->h2d, c->ev_free[1][slot], 0));
    cudaEvent_t c0 = get_event(c), c1 = get_event(c);
    CK(cudaEventRecord(c0, c->h2d));
    u8 *ha = nullptr, *da = nullptr; u64 len = 0;
    for (u64 u = u0; u < u1; ++u) {
      u8* h = c->h_store + (u64)su[u] * c->blk;
      u8* d = c->staging[1][slot] + (u - u0) * c->blk;
      if (len && h == ha + len && d == da + len) len += c->blk;
      else {
        if (len) { CK(cudaMemcpyAsync(da, ha, len, cudaMemcpyHostToDevice, c->h2d)); op.copy_bytes += len; }
        ha = h; da = d; len = c->blk;
      }
    }
    if (len) { CK(cudaMemcpyAsync(da, ha, len, cudaMemcpyHostToDevice, c->h2d)); op.copy_bytes += len; }
    CK(cudaEventRecord(c1, c->h2d));
    op.t_copy.push_back({c0, c1});
    CK(cudaEventRecord(c->ev_ready[1][slot], c->h2d));
    CK(cudaStreamWaitEvent(c->scatter, c->ev_ready[1][slot], 0));
    u32 nf = 0;
    while (fi < flips.size() && flips[fi].first < u1) {
      c->h_flip[flip_base + nf++] = (flips[fi].first - u0) * c->blk + flips[fi].second;
      ++fi;
    }
    if (nf) {
      CK(to_dev(c, c->scatter, c->d_flip + flip_base, c->h_flip + flip_base, (u64)nf * 8));
      k_bitflip<<<(nf + 63) / 64, 64, 0, c->scatter>>>(c->staging[1][slot], c->d_flip + flip_base, nf);
      CKL();
      c->st.kernel_launches++;
      flip_base += nf;
    }
    size_t je = ji;                                        // the items whose staged block lives in this chunk
    while (je < items.size() && items[je].first / c->chunk_blocks == ci) ++je;
    for (size_t j0 = ji; j0 < je; j0 += c->chunk_blocks) { // the partial-sum buffer holds chunk_blocks items per launch
      const u32 m = (u32)std::min<u64>(c->chunk_blocks, je - j0);
      cudaEvent_t t0 = get_event(c), t1 = get_event(c);
      CK(cudaEventRecord(t0, c->scatter));
      launch_move<MV_SCATTER>(c, c->scatter, c->staging[1][slot], c->d_phys[1], c->part[1][slot], m, c->d_iw + j0, c->d_ispos + j0);
      CKL();
      CK(cudaEventRecord(t1, c->scatter));
      op.t_kernel.push_back({t0, t1});
      op.launches++;
      k_block_digest<<<warps_grid(m), 256, 0, c->scatter>>>(c->part[1][slot], c->d_phys[1], c->d_dtmp[1], c->d_etmp[1], m, c->G, c->d_iw + j0);
      CKL();
      c->st.kernel_launches++;
    }
    ji = je;
    CK(cudaEventRecord(c->ev_free[1][slot], c->scatter));
    c->slot_used[1][slot] = true;
  }
  return restore_opened(c, n_served);
}
