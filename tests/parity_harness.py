"""GPU-vs-oracle parity harness: drives librc (CUDA, through the C ABI) and the oracle over the
same seeded waves and compares every observable after every call, element by element.

The oracle works on a host mirror of the pool taken with tensor.cpu() -- a path that does not
touch the kernels under test.  Freed blocks are poisoned on both sides between offload and
restore (DESIGN R5) so a restore that did not really read the host copy is caught.
"""
import numpy as np
import torch

from oracle import rco
from paper_2606_01387_b200 import rc, workloads as W


class Pair:
    def __init__(self, wl, host_store_bytes, chunk_blocks=None, staging_chunks=2, mover=rc.MOVER_AUTO,
                 grid_ctas=0, oracle_host_store_bytes=None, max_events=1 << 17, seed=None, dedup=False, copies=(), direct_offload=False, layer_major=False):
        g = wl.geom
        self.wl, self.g = wl, g
        dev = torch.device("cuda:0")
        self.pool_t = W.pool_torch(g, dev, seed)
        v = self.pool_t.view(2 * g.layers, g.pool_blocks, g.page_bytes)
        for src, dst in copies:                            # identical content in different physical blocks
            v[:, dst, :] = v[:, src, :]
        torch.cuda.synchronize()
        self.pool_h = self.pool_t.cpu().numpy()
        self.fill_t = torch.zeros(g.pool_blocks, dtype=torch.uint8, device=dev)
        self.fill_h = np.zeros(g.pool_blocks, np.uint8)
        self.o = rco.Oracle(g.layers, g.kv_heads, g.head_dim, g.elem_bytes, g.block_size, g.pool_blocks,
                            self.pool_h, self.fill_h,
                            host_store_bytes if oracle_host_store_bytes is None else oracle_host_store_bytes)
        self.r = rc.RC(g.layers, g.kv_heads, g.head_dim, g.elem_bytes, g.block_size, g.pool_blocks,
                       self.pool_t, self.fill_t, host_store_bytes,
                       staging_chunk_bytes=(chunk_blocks * g.blk_bytes) if chunk_blocks else None,
                       staging_chunks=staging_chunks, mover=mover, grid_ctas=grid_ctas, max_events=max_events, dedup=dedup, direct_offload=direct_offload,
                       layer_major=layer_major)
        if dedup:
            assert self.o.set_dedup(True) == 0
        if layer_major:
            assert self.o.set_layer_major(True) == 0
        self.dedup = dedup
        self.view_h = self.pool_h.reshape(2 * g.layers, g.pool_blocks, g.page_bytes)
        self.view_t = self.pool_t.view(2 * g.layers, g.pool_blocks, g.page_bytes)

    def close(self):
        self.r.close()
        self.o.close()

    # ---- inputs, applied identically to both sides -------------------------------------------
    def set_fill(self, ids, vals):
        self.fill_h[ids] = vals
        self.fill_t[torch.from_numpy(np.asarray(ids).astype(np.int64)).cuda()] = torch.from_numpy(
            np.asarray(vals, np.uint8)).cuda()
        torch.cuda.synchronize()

    def poison_free(self):
        used, _ = self.o.pool_state()
        free = np.nonzero(used == 0)[0]
        self.view_h[:, free, :] = W.POISON
        if free.size:
            self.view_t[:, torch.from_numpy(free.astype(np.int64)).cuda(), :] = W.POISON
            torch.cuda.synchronize()          # torch's stream is not ordered against the library's non-blocking streams

    def logical(self, cid):
        """Claim-logical KV [block][page g][bytes] read with torch indexing (not with librc)."""
        bt = self.r.claim_blocks(cid)
        idx = torch.from_numpy(bt.astype(np.int64)).cuda()
        return self.view_t[:, idx, :].permute(1, 0, 2).contiguous().cpu().numpy()

    # ---- comparisons ---------------------------------------------------------------------------
    def check_claims(self, ids, what, digests=True, host=False):
        for cid in ids:
            a, b = self.o.claim_info(cid), self.r.claim_info(cid)
            assert a == b, "%s: claim_info differs for %x: oracle %r, cuda %r" % (what, cid, a, b)
            if a is None:
                continue
            assert np.array_equal(self.o.claim_blocks(cid), self.r.claim_blocks(cid)), "%s: table %x" % (what, cid)
            if digests:
                (da, ea), (db, eb) = self.o.claim_digests(cid, both=True), self.r.claim_digests(cid, both=True)
                assert np.array_equal(da, db), "%s: digests d %x" % (what, cid)
                assert np.array_equal(ea, eb), "%s: digests e %x" % (what, cid)
            if host:
                ha, hb = self.o.host_read(cid), self.r.host_read(cid)
                assert ha.size == hb.size and np.array_equal(ha, hb), "%s: host bytes %x" % (what, cid)

    def check_pool_state(self, what, bytes_too=True):
        ua, ra = self.o.pool_state()
        ub, rb = self.r.pool_state()
        assert np.array_equal(ua, ub), "%s: used[] differs at %r" % (what, np.nonzero(ua != ub)[0][:8])
        assert np.array_equal(ra, rb), "%s: ref[] differs at %r" % (what, np.nonzero(ra != rb)[0][:8])
        assert np.array_equal(self.fill_h, self.fill_t.cpu().numpy()), "%s: fill[] differs" % what
        if bytes_too:                                        # raw pool bytes of every live block
            live = np.nonzero(ua == 1)[0]
            for s in range(0, live.size, 256):
                ix = live[s:s + 256]
                got = self.view_t[:, torch.from_numpy(ix.astype(np.int64)).cuda(), :].cpu().numpy()
                assert np.array_equal(got, self.view_h[:, ix, :]), "%s: pool bytes differ in blocks %r.." % (what, ix[:4])

    def check_events(self, what):
        ea, eb = self.o.outcomes(), self.r.outcomes()
        assert ea.size == eb.size, "%s: %d oracle events, %d cuda events" % (what, ea.size, eb.size)
        if ea.size and not np.array_equal(ea, eb):
            bad = [i for i in range(ea.size) if ea[i] != eb[i]][:4]
            raise AssertionError("%s: events differ at %r: %r vs %r" % (what, bad, ea[bad], eb[bad]))
        return ea

    # ---- one wave, every step compared ---------------------------------------------------------
    def run_wave(self, wave, restore_batches=None, faults=None, fault_flags=0, check_bytes=True, release=True):
        wl = self.wl
        cl = [wl.claims[k] for k in wave.claim_idx]
        ids = [c.claim_id for c in cl]
        self.set_fill(wave.fill_ids, wave.fill_val)
        assert self.o.mark_used(wave.used_ids) == 0 and self.r.mark_used(wave.used_ids) == 0
        args = (ids, [c.P for c in cl], [c.N for c in cl], wave.bt_off, wave.bt_ids)
        sa, sb = self.o.accept(*args), self.r.accept(*args)
        assert np.array_equal(sa, sb), "accept status %r vs %r" % (sa, sb)
        self.check_claims(ids, "accept", digests=False)
        sa, sb = self.o.materialize(ids), self.r.materialize(ids)
        assert np.array_equal(sa, sb), "materialize status %r vs %r" % (sa, sb)
        self.check_claims(ids, "materialize", digests=False)
        before = {c.claim_id: self.logical(c.claim_id) for c, s in zip(cl, sa) if s == 0} if check_bytes else {}
        sa, sb = self.o.offload(ids), self.r.offload(ids)
        assert np.array_equal(sa, sb), "offload status %r vs %r" % (sa, sb)
        self.check_claims(ids, "offload", host=check_bytes)
        self.check_pool_state("offload", bytes_too=False)
        self.poison_free()
        fl = wave.faults if faults is None else faults
        assert self.o.set_faults(fl, fault_flags) == 0 and self.r.set_faults(fl, fault_flags) == 0
        st_r = []
        for batch in (restore_batches or [ids]):
            sa, sb = self.o.restore(batch), self.r.restore(batch)
            assert np.array_equal(sa, sb), "restore status %r vs %r" % (sa, sb)
            st_r.extend(int(x) for x in sa)
            self.check_claims(batch, "restore")
            self.check_pool_state("restore", bytes_too=check_bytes)
        for c in cl:                                         # bit-exact round trip of the claim-logical view
            info = self.r.claim_info(c.claim_id)
            if check_bytes and info["state"] == 4:
                assert np.array_equal(self.logical(c.claim_id), before[c.claim_id][: info["nb"]]), \
                    "round trip differs for claim %x" % c.claim_id
        ev = self.check_events("wave")
        sa, sb = self.o.stats(), self.r.stats()
        assert sa["generic_failures"] == sb["generic_failures"] and sa["host_used"] == sb["host_used_bytes"]
        assert self.o.link_bytes() == (sb["bytes_d2h"], sb["bytes_h2d"]), "link bytes: oracle %r, cuda %r" % (
            self.o.link_bytes(), (sb["bytes_d2h"], sb["bytes_h2d"]))
        if release:
            sa, sb = self.o.release(ids), self.r.release(ids)
            assert np.array_equal(sa, sb)
            self.check_pool_state("release", bytes_too=False)
        return ev, st_r
