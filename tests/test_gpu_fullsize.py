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
