"""Parity at BASELINE.json's full size, in the launch configuration bench.py times (configs[1]: Llama-3-8B KV
shape, 8192-block = 16 GiB pool, 2 GiB staging chunks, default TMA mover, restore(k) overlapped with
offload(k+1)).  The oracle cannot replay 71 GiB in seconds, so: sampled outputs it can compute one by one
(block digests and chains of sampled claims from the host-store bytes), properties that hold at any size
(bit-exact round trip against a torch gather taken before the offload, host-store bytes equal to that gather,
validator-accepted event stream, statuses and M from the recipe)."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

from oracle import rco, validator as V
from paper_2606_01387_b200 import rc, workloads as W


def test_config1_full_size_bench_configuration():
    wl = W.make_workload(1)
    g = wl.geom
    dev = torch.device("cuda:0")
    host = g.pool_bytes
    waves = W.plan_waves(wl, host // 4, pool_blocks=g.pool_blocks // 4)[:4]
    pool = W.pool_torch(g, dev)
    fill = torch.zeros(g.pool_blocks, dtype=torch.uint8, device=dev)
    r = rc.RC(g.layers, g.kv_heads, g.head_dim, g.elem_bytes, g.block_size, g.pool_blocks, pool, fill, host,
              staging_chunk_bytes=2 << 30, max_claims=1024)
    view = pool.view(2 * g.layers, g.pool_blocks, g.page_bytes)
    rng = np.random.default_rng(5)

    def logical(cid):
        idx = torch.from_numpy(r.claim_blocks(cid).astype(np.int64)).to(dev)
        return view[:, idx, :].permute(1, 0, 2).contiguous()          # [block][g][page] on the GPU (torch, not librc)

    def admit(w):
        cl = [wl.claims[k] for k in w.claim_idx]
        ids = [c.claim_id for c in cl]
        fill[torch.from_numpy(w.fill_ids.astype(np.int64)).to(dev)] = torch.from_numpy(w.fill_val).to(dev)
        assert r.mark_used(w.used_ids) == 0
        assert not r.accept(ids, [c.P for c in cl], [c.N for c in cl], w.bt_off, w.bt_ids).any()
        assert not r.materialize(ids).any()
        for c in cl:
            assert r.claim_info(c.claim_id)["M"] == c.M
        before = {c.claim_id: logical(c.claim_id) for c in cl}
        return cl, ids, before

    def check_offloaded(cl, before):
        for c in [cl[i] for i in rng.choice(len(cl), 3, replace=False)]:
            info = r.claim_info(c.claim_id)
            hb = r.host_read(c.claim_id)
            assert np.array_equal(hb, before[c.claim_id][: info["nb"]].cpu().numpy().reshape(-1))   # host bytes = gather
            d, e = r.claim_digests(c.claim_id, both=True)
            for i in rng.choice(info["nb"], min(4, info["nb"]), replace=False):                    # oracle, block by block
                assert int(d[i]) == rco.block_digest(hb[i * g.blk_bytes:(i + 1) * g.blk_bytes], 2 * g.layers, 0)
                assert int(e[i]) == rco.block_digest(hb[i * g.blk_bytes:(i + 1) * g.blk_bytes], 2 * g.layers, 1)
            assert info["chain"] == rco.chain_of(c.claim_id, d)

    def check_restored(cl, st, before):
        faulted = {c.claim_id for c in cl if c.fault}
        for c, s in zip(cl, st):
            info = r.claim_info(c.claim_id)
            if c.claim_id in faulted:
                assert s == rc.ST_RESTORE_FAILED and info["state"] == 5
            else:
                assert s == rc.ST_OK and info["state"] == 4
                assert torch.equal(logical(c.claim_id), before[c.claim_id][: info["nb"]])          # bit-exact round trip

    events = []
    cl, ids, before = admit(waves[0])
    assert not r.offload(ids).any()
    check_offloaded(cl, before)
    for k in range(len(waves)):
        nxt = admit(waves[k + 1]) if k + 1 < len(waves) else None
        used, _ = r.pool_state()
        free = torch.from_numpy(np.nonzero(used == 0)[0].astype(np.int64)).to(dev)
        view[:, free, :] = W.POISON                                                               # restore must read the host copy
        torch.cuda.synchronize()              # torch's stream is not ordered against the library's non-blocking streams
        assert r.set_faults([(c.claim_id,) + c.fault for c in cl if c.fault]) == 0
        r.restore_begin(ids)
        if nxt:
            r.offload_begin(nxt[1])
            assert not r.wait(0).any()
        st = r.wait(1)
        check_restored(cl, st, before)
        if nxt:
            check_offloaded(nxt[0], nxt[2])
        events.append(r.outcomes())
        assert not r.release(ids).any()
        if nxt:
            cl, ids, before = nxt
    ev = np.concatenate(events)
    ok, why = V.validate(ev)
    assert ok, why
    assert list(ev["seq"]) == list(range(len(ev)))
    s = r.stats()
    assert s["gather_launches"] > 0 and s["bytes_d2h"] == s["gather_blocks"] * g.blk_bytes
    r.close()


# ---- configs[2], [3], [4] at BASELINE.json's full size, in bench.py's launch configuration ----------------------------
# (2 GiB staging chunks, default TMA movers, restore(k) overlapped with offload(k+1) and offload(k+2), waves placed as
# bench.py places them).  What is checked, per wave: statuses and M from the recipe; for sampled claims (always the largest one, so the
# claim spans the most staging chunks) sampled blocks -- first, last, both sides of every chunk boundary, random -- are
# compared byte for byte between a torch copy taken before the offload, the pinned host store (rc_host_store view) and the
# restored pool; their digests d, e and the claim's chain are recomputed by the oracle from the host bytes; every block of
# every claim is compared through a torch fingerprint (two wrapping int64 sums) taken before the offload and after the
# restore, with all free blocks poisoned in between; the event stream is accepted by the oracle's validator.
import ctypes
import hashlib
import os
from concurrent.futures import ThreadPoolExecutor


def _need(dev_bytes, host_bytes):
    free, _ = torch.cuda.mem_get_info()
    avail = os.sysconf("SC_PAGE_SIZE") * os.sysconf("SC_AVPHYS_PAGES")
    if free < dev_bytes:
        pytest.skip("needs %.0f GB of device memory, %.0f GB free" % (dev_bytes / 1e9, free / 1e9))
    if avail < host_bytes:
        pytest.skip("needs %.0f GB of host memory for the pinned store, %.0f GB available" % (host_bytes / 1e9, avail / 1e9))


class FullSize:
    def __init__(self, index, wave_frac, host_bytes, max_claims_per_wave=None, dedup=False, n_waves=3, layer_major=False):
        self.wl = wl = W.make_workload(index)
        self.g = g = wl.geom
        _need(g.pool_bytes + (14 << 30), host_bytes + (12 << 30))
        self.dev = dev = torch.device("cuda:0")
        region = g.pool_blocks // wave_frac
        self.waves = W.plan_waves(wl, host_bytes // 3, pool_blocks=region, max_claims_per_wave=max_claims_per_wave)[:n_waves]
        for wi, w in enumerate(self.waves):                       # bench.py's placement: two alternating top regions
            base = np.uint32(g.pool_blocks - (1 + wi % 2) * region)
            w.bt_ids, w.used_ids, w.fill_ids = w.bt_ids + base, w.used_ids + base, w.fill_ids + base
        self.pool = W.pool_torch(g, dev)
        self.fill = torch.zeros(g.pool_blocks, dtype=torch.uint8, device=dev)
        n_max = max(len(w.claim_idx) for w in self.waves)
        self.r = rc.RC(g.layers, g.kv_heads, g.head_dim, g.elem_bytes, g.block_size, g.pool_blocks, self.pool, self.fill,
                       host_bytes, staging_chunk_bytes=2 << 30, staging_chunks=2, max_claims=max(1024, 4 * n_max),
                       max_table_entries=max(4 * g.pool_blocks, 1 << 16), max_events=max(1 << 16, 16 * n_max), dedup=dedup,
                       layer_major=layer_major)
        self.lm = layer_major
        self.view = self.pool.view(2 * g.layers, g.pool_blocks, g.page_bytes)
        self.rng = np.random.default_rng(100 + index)
        wgen = torch.Generator(device=dev)
        wgen.manual_seed(5)
        self.wts = torch.randint(-(1 << 62), 1 << 62, (2 * g.layers, 1, g.page_bytes // 8), dtype=torch.int64, device=dev,
                                 generator=wgen) | 1
        self.chunk_blocks = (2 << 30) // g.blk_bytes
        self.events = []

    def close(self):
        import gc
        self.r.close()
        del self.pool, self.view, self.fill, self.wts
        self.events = []
        gc.collect()
        torch.cuda.empty_cache()

    def fingerprint(self, blocks):
        """Two wrapping int64 sums per block over all its pages, on the GPU with torch (not with librc)."""
        out = []
        idx = torch.from_numpy(np.asarray(blocks).astype(np.int64)).to(self.dev)
        step = max(1, (256 << 20) // self.g.blk_bytes)
        for s in range(0, idx.numel(), step):
            x = self.view[:, idx[s:s + step], :].view(torch.int64)
            out.append(torch.stack([x.sum(dim=(0, 2)), (x * self.wts).sum(dim=(0, 2))], 1))
        return torch.cat(out) if out else torch.zeros((0, 2), dtype=torch.int64, device=self.dev)

    def sample_blocks(self, nb):
        cb = self.chunk_blocks
        s = {0, nb - 1} | {int(x) for x in self.rng.integers(0, nb, 3)}
        for b in range(cb, nb, cb):
            s |= {b - 1, b}
        return sorted(x for x in s if 0 <= x < nb)

    def admit(self, w):
        wl, r = self.wl, self.r
        cl = [wl.claims[k] for k in w.claim_idx]
        ids = [c.claim_id for c in cl]
        self.fill[torch.from_numpy(w.fill_ids.astype(np.int64)).to(self.dev)] = torch.from_numpy(w.fill_val).to(self.dev)
        torch.cuda.synchronize()
        assert r.mark_used(w.used_ids) == 0
        assert not r.accept(ids, [c.P for c in cl], [c.N for c in cl], w.bt_off, w.bt_ids).any()
        st = r.materialize(ids)
        assert [int(s) for s in st] == [0 if c.M >= c.N else 1 for c in cl]                 # predicate from the recipe
        served = [c for c in cl if c.M >= c.N]
        info = {c.claim_id: r.claim_info(c.claim_id) for c in served}
        assert all(info[c.claim_id]["M"] == c.M for c in served)
        tabs = {c.claim_id: r.claim_blocks(c.claim_id)[: info[c.claim_id]["nb"]] for c in served}
        fp = {cid: self.fingerprint(t) for cid, t in tabs.items()}
        big = max(served, key=lambda c: info[c.claim_id]["nb"])
        pick = {big.claim_id} | {served[i].claim_id for i in self.rng.choice(len(served), min(2, len(served)), replace=False)}
        keep = {}
        for cid in pick:
            S = self.sample_blocks(len(tabs[cid]))
            ix = torch.from_numpy(tabs[cid][S].astype(np.int64)).to(self.dev)
            keep[cid] = (S, self.view[:, ix, :].permute(1, 0, 2).contiguous().cpu().numpy())   # [sample][g][page]
        return dict(cl=cl, ids=ids, served=served, fp=fp, keep=keep, nb={k: v["nb"] for k, v in info.items()})

    def check_offloaded(self, a, st):
        g, r = self.g, self.r
        assert [int(s) for s in st] == [0 if c.M >= c.N else 3 for c in a["cl"]]
        for cid, (S, want) in a["keep"].items():
            info = r.claim_info(cid)
            assert info["state"] == 3 and info["nb"] == a["nb"][cid] and info["host_bytes"] == info["nb"] * g.blk_bytes
            d, e = r.claim_digests(cid, both=True)
            whole = r.host_read(cid).reshape(2 * g.layers, info["nb"], g.page_bytes) if self.lm else None   # [g][block][page]
            for j, i in enumerate(S):
                hb = np.ascontiguousarray(whole[:, i, :]).reshape(-1) if self.lm else r.host_store(cid, i)
                assert hb is not None and np.array_equal(hb, want[j].reshape(-1)), "host bytes of claim %x block %d" % (cid, i)
                assert int(d[i]) == rco.block_digest(hb, 2 * g.layers, 0) and int(e[i]) == rco.block_digest(hb, 2 * g.layers, 1)
            assert info["chain"] == rco.chain_of(cid, d)

    def check_restored(self, a, st):
        r = self.r
        for c, s in zip(a["cl"], st):
            if c.M < c.N:
                assert s == rc.ST_BAD_STATE                                   # never materialized: nothing to restore
                continue
            info = r.claim_info(c.claim_id)
            if c.fault:
                assert s == rc.ST_RESTORE_FAILED and info["state"] == 5 and info["n_table"] == 0
                continue
            assert s == rc.ST_OK and info["state"] == 4 and info["n_table"] == a["nb"][c.claim_id]
            bt = r.claim_blocks(c.claim_id)
            assert torch.equal(self.fingerprint(bt), a["fp"][c.claim_id]), "round trip of claim %x" % c.claim_id
            if c.claim_id in a["keep"]:
                S, want = a["keep"][c.claim_id]
                ix = torch.from_numpy(bt[S].astype(np.int64)).to(self.dev)
                assert np.array_equal(self.view[:, ix, :].permute(1, 0, 2).contiguous().cpu().numpy(), want)

    def poison_free(self):
        used, _ = self.r.pool_state()
        free = torch.from_numpy(np.nonzero(used == 0)[0].astype(np.int64)).to(self.dev)
        for s in range(0, free.numel(), 4096):
            self.view[:, free[s:s + 4096], :] = W.POISON
        torch.cuda.synchronize()

    def run(self, extra_faults=(), flags=0):
        """bench.py's pipelined schedule: while restore(k) is in flight, offload(k+1) and offload(k+2) run back to back
        (two open offloads); rc_wait(0) completes offload(k) before restore(k) begins."""
        r = self.r
        adm = [self.admit(w) for w in self.waves[:2]]
        st_o = [r.offload_begin(a["ids"]) for a in adm]
        for k in range(len(self.waves)):
            a = adm[k]
            r.wait(0)                                                        # completes offload(k)
            self.check_offloaded(a, st_o[k])
            if k + 2 < len(self.waves):
                adm.append(self.admit(self.waves[k + 2]))                    # the region offload(k) has just left
            self.poison_free()                                               # restore must read the host copy
            faults = [(c.claim_id,) + c.fault for c in a["cl"] if c.fault] + list(extra_faults)
            assert r.set_faults(faults, flags) == 0
            st_r = r.restore_begin(a["ids"])
            if k + 2 < len(self.waves):
                st_o.append(r.offload_begin(adm[k + 2]["ids"]))              # open: offload(k+1), offload(k+2)
            r.wait(1)
            self.check_restored(a, st_r)
            self.events.append(r.outcomes())
            assert not r.release(a["ids"]).any()
        ev = np.concatenate(self.events)
        ok, why = V.validate(ev)
        assert ok, why
        assert list(ev["seq"]) == list(range(len(ev)))
        return ev


def test_config1_full_size_two_open_offloads():
    """configs[1] (the workload bench.py's `value` is quoted on) in bench.py's default launch configuration: waves of 1/8 of
    the 16 GiB pool in two alternating top regions, 2 GiB staging chunks, two open offloads ahead of the restore."""
    fs = FullSize(1, wave_frac=8, host_bytes=16 << 30, n_waves=6)
    ev = fs.run()
    n_fault = sum(1 for w in fs.waves for k in w.claim_idx if fs.wl.claims[k].fault)
    s = fs.r.stats()
    assert s["claims_refused"] == n_fault and int((ev["code"] == 8).sum()) == n_fault
    assert s["bytes_d2h"] == s["gather_blocks"] * fs.g.blk_bytes and s["bytes_h2d"] <= s["bytes_d2h"]
    fs.close()


def test_config2_llama70b_full_size():
    """Llama-3-70B shape: 20000-block = 105 GB pool, 5 MiB blocks, Zipf-shared prefixes (ref > 1), 10 % under-materialized."""
    fs = FullSize(2, wave_frac=8, host_bytes=32 << 30)
    ev = fs.run()
    s = fs.r.stats()
    assert s["bytes_d2h"] == s["gather_blocks"] * fs.g.blk_bytes and s["claims_refused"] == sum(
        1 for w in fs.waves for k in w.claim_idx if fs.wl.claims[k].fault)
    assert any(fs.wl.claims[k].shared for w in fs.waves for k in w.claim_idx)
    fs.close()


def test_config2_full_size_dedup_link_bytes_equal_distinct_contents():
    """Same pool, content-addressed store: the D2H link bytes of a wave equal blk x the number of distinct block contents
    among the blocks its claims offload, counted here with SHA-256 over bytes read back with torch."""
    fs = FullSize(2, wave_frac=8, host_bytes=16 << 30, max_claims_per_wave=4, dedup=True, n_waves=2)
    g, r = fs.g, fs.r
    w = fs.waves[0]
    ok = [j for j, k in enumerate(w.claim_idx) if fs.wl.claims[k].M >= fs.wl.claims[k].N]
    t0, t1 = (w.bt_ids[w.bt_off[j]:w.bt_off[j + 1]] for j in ok[:2])
    src = torch.from_numpy(t0[5:45].astype(np.int64)).to(fs.dev)                # identical content in different physical
    dst = torch.from_numpy(t1[-60:-20].astype(np.int64)).to(fs.dev)             # blocks of two claims, besides the
    fs.view[:, dst, :] = fs.view[:, src, :]                                      # physically shared prefix blocks
    torch.cuda.synchronize()
    a = fs.admit(w)
    tabs = [r.claim_blocks(c.claim_id)[: a["nb"][c.claim_id]] for c in a["served"]]
    blocks = np.concatenate(tabs)

    def sha(b):
        ix = torch.tensor([int(b)], device=fs.dev)
        return hashlib.sha256(fs.view[:, ix, :].cpu().numpy().tobytes()).digest()
    with ThreadPoolExecutor(8) as ex:
        digs = list(ex.map(sha, np.unique(blocks)))
    by_block = dict(zip([int(b) for b in np.unique(blocks)], digs))
    distinct = len({by_block[int(b)] for b in blocks})
    assert distinct <= len(blocks) - 40
    st = r.offload(a["ids"])
    fs.check_offloaded(a, st)
    s = r.stats()
    assert s["bytes_d2h"] == distinct * g.blk_bytes and s["host_used_bytes"] == distinct * g.blk_bytes
    assert s["gather_blocks"] == len(blocks)
    fs.poison_free()
    st_r = r.restore(a["ids"])
    fs.check_restored(a, st_r)
    n_ok = sum(1 for c in a["served"] if not c.fault)
    assert r.stats()["bytes_h2d"] <= distinct * g.blk_bytes + sum(a["nb"][c.claim_id] for c in a["served"] if c.fault) * g.blk_bytes
    assert n_ok > 0 and V.validate(r.outcomes())[0]
    fs.close()


def test_config3_fp8_full_size_with_decoys():
    """fp8 shape: 65536-block pool, 16 KiB pages (the 8 KiB-tile TMA instantiation on a 16 KiB page), ~200 short claims per
    wave, 5 % real faults plus decoy fault entries (never-accepted ids, id 0 under the flag, accepted-but-not-restored
    claims) that must change nothing."""
    fs = FullSize(3, wave_frac=8, host_bytes=32 << 30)
    ev = fs.run(extra_faults=fs.wl.decoys, flags=rc.FAULT_ALLOW_UNCLAIMED)
    in_waves = {fs.wl.claims[k].claim_id: fs.wl.claims[k] for w in fs.waves for k in w.claim_idx}
    failed = {int(e["claim_id"]) for e in ev if int(e["code"]) == 8}
    assert failed == {cid for cid, c in in_waves.items() if c.fault} and len(failed) > 5
    assert all(int(e["claim_id"]) in in_waves for e in ev)                     # no decoy id ever appears in the stream
    n_unclaimed = sum(1 for d in fs.wl.decoys if d[0] == 0)
    assert fs.r.stats()["generic_failures"] == n_unclaimed * len(fs.waves)     # counters, never outcomes
    fs.close()


def test_config4_long_context_full_size_interleaved():
    """Long context: 61440-block = 120 GiB pool, claims of 2048-8192 blocks with partial materialization: every claim
    spans 2-8 staging chunks; batches interleaved begin/wait as BASELINE.json configs[4] states."""
    fs = FullSize(4, wave_frac=4, host_bytes=64 << 30, max_claims_per_wave=8, n_waves=3)
    assert max(fs.wl.claims[k].M for w in fs.waves for k in w.claim_idx) > 2 * fs.chunk_blocks * fs.g.block_size   # > 2 staging chunks
    ev = fs.run()
    n = sum(len(w.claim_idx) for w in fs.waves)
    assert int((ev["code"] == 6).sum()) == n and fs.r.stats()["claims_restored"] == n
    fs.close()


def test_config1_full_size_layer_major():
    """configs[1] in bench.py's launch configuration with rc_config.layer_major: the host copy is [g][block][page]; sampled
    blocks are cut out of it by that layout and must equal the torch copy taken before the offload, their digests the
    oracle's; round trip, fingerprints, stream as in every other full-size run."""
    fs = FullSize(1, wave_frac=8, host_bytes=16 << 30, n_waves=4, layer_major=True)
    ev = fs.run()
    s = fs.r.stats()
    assert s["bytes_d2h"] == s["gather_blocks"] * fs.g.blk_bytes and int((ev["code"] == 6).sum()) > 0
    fs.close()
