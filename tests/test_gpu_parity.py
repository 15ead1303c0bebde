"""GPU parity: librc (CUDA, through the C ABI) against the oracle, bit-exact, on BASELINE.json
configs[0..4] (configs 1-4 at reduced unit counts so the oracle finishes in seconds; same recipe).
Compared after every call: statuses, claim info, block tables, digests, chains, host-store
bytes, allocator state, fill, raw pool bytes of live blocks, the claim-logical round trip and the
event stream (P:L27 order per claim, batch-major across claims)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import rco, validator as V
from paper_2606_01387_b200 import rc, workloads as W
from parity_harness import Pair
from shared_tiny import make_shared_tiny

GOLD = [l.split("#")[0].strip() for l in open(__file__.rsplit("/", 1)[0] + "/golden/event_orders.txt")]
GOLD = {l.split(":")[0].strip(): [x.strip() for x in l.split(":")[1].split(",")] for l in GOLD if l}


def names(ev, cid):
    return [rco.EV_NAMES[int(e["code"])] for e in ev if int(e["claim_id"]) == cid]


@pytest.mark.parametrize("mover", [rc.MOVER_LDG, rc.MOVER_TMA])
@pytest.mark.parametrize("kind", [W.FK_BITFLIP, W.FK_XFER_ERROR])
@pytest.mark.parametrize("chunk_blocks", [5, 64])
def test_tiny_full_parity(mover, kind, chunk_blocks):
    wl = W.make_workload(0)
    p = Pair(wl, 1 << 30, chunk_blocks=chunk_blocks, mover=mover)
    wave = W.plan_waves(wl, 1 << 30)[0]
    faults = [(cid, kind, prm) for cid, _, prm in wave.faults]
    ev, st_r = p.run_wave(wave, faults=faults)
    ok, why = V.validate(ev)
    assert ok, why
    for k, c in enumerate(wl.claims):
        got = names(ev, c.claim_id)
        if k == 6:
            assert got == ["ACCEPTED"] and st_r[k] == rc.ST_BAD_STATE
        elif k == 3:
            assert got == GOLD["failure_path"] and st_r[k] == rc.ST_RESTORE_FAILED     # P:L27, exact
        else:
            assert got == GOLD["success_path"] and st_r[k] == rc.ST_OK
    p.close()


def _run_config(index, n_claims, pool_blocks, host_bytes, chunk_blocks, mover=rc.MOVER_AUTO, flags=0, scale=None,
                sub=None):
    kw = {} if scale is None else {"scale": scale}
    wl = W.make_workload(index, n_claims=n_claims, pool_blocks=pool_blocks, **kw)
    p = Pair(wl, host_bytes, chunk_blocks=chunk_blocks, mover=mover)
    evs = []
    for wave in W.plan_waves(wl, host_bytes):
        ids = [wl.claims[k].claim_id for k in wave.claim_idx]
        faults = wave.faults + (wl.decoys if flags else [])
        batches = [ids[i:i + sub] for i in range(0, len(ids), sub)] if sub else None
        ev, _ = p.run_wave(wave, restore_batches=batches, faults=faults, fault_flags=flags)
        ok, why = V.validate(ev)
        assert ok, why
        evs.append(ev)
    p.close()
    return wl, evs


@pytest.mark.parametrize("mover", [rc.MOVER_LDG, rc.MOVER_TMA])
def test_config1_llama8b_reduced(mover):
    wl, evs = _run_config(1, 6, 768, 2 << 30, chunk_blocks=37, mover=mover)
    assert sum(len(e) for e in evs) > 0


def test_config2_llama70b_shared_prefixes_reduced():
    # Zipf-shared prefix groups: shared physical blocks (ref > 1), duplicated in the host store,
    # restored in sub-batches that fit the free pool
    _run_config(2, 4, 1300, 6 << 30, chunk_blocks=50, sub=2)


def test_config3_fp8_decoys_reduced():
    wl, evs = _run_config(3, 80, 2048, 4 << 30, chunk_blocks=100, flags=rc.FAULT_ALLOW_UNCLAIMED)
    ev = np.concatenate(evs)
    failed = {int(e["claim_id"]) for e in ev if int(e["code"]) == 8}
    real = {c.claim_id for c in wl.claims if c.fault}
    assert failed == real                   # decoys (never-accepted ids, id 0, not-restored claims) changed nothing


def test_config4_long_context_interleaved_reduced():
    # batches of 8 claims; restore of batch k overlapped with the offload of batch k+1 (begin/wait),
    # compared with the oracle making the same calls synchronously in begin order
    wl = W.make_workload(4, n_claims=24, pool_blocks=2048, scale=64)
    host = 3 << 30
    p = Pair(wl, host, chunk_blocks=64)
    o, r = p.o, p.r
    B = wl.batch
    batches = [list(range(i, min(i + B, len(wl.claims)))) for i in range(0, len(wl.claims), B)]
    waves = W.plan_waves(wl, host, max_claims_per_wave=B)
    assert [w.claim_idx for w in waves] == batches

    def admit(wave):
        cl = [wl.claims[k] for k in wave.claim_idx]
        ids = [c.claim_id for c in cl]
        used, _ = o.pool_state()
        free = np.nonzero(used == 0)[0].astype(np.uint32)
        assert free.size >= wave.used_ids.size
        remap = np.zeros(wl.geom.pool_blocks, np.uint32)       # place the wave's tables on currently free blocks
        remap[wave.used_ids] = free[: wave.used_ids.size]
        bt = remap[wave.bt_ids]
        p.set_fill(remap[wave.fill_ids], wave.fill_val)
        assert o.mark_used(remap[wave.used_ids]) == 0 and r.mark_used(remap[wave.used_ids]) == 0
        args = (ids, [c.P for c in cl], [c.N for c in cl], wave.bt_off, bt)
        assert np.array_equal(o.accept(*args), r.accept(*args))
        assert np.array_equal(o.materialize(ids), r.materialize(ids))
        return ids

    prev = None
    for wave in waves:
        ids = admit(wave)
        if prev is None:
            assert np.array_equal(o.offload(ids), r.offload(ids))
        else:
            # cuda: both in flight at once; the restore's plan takes effect at its _begin, the offload at rc_wait(0), the
            # restore's verdicts and records at rc_wait(1) (rc.h split forms) -- the oracle makes exactly these calls
            o.restore_begin(prev)
            r.restore_begin(prev)
            r.offload_begin(ids)
            sa_o, sb_o = o.offload(ids), r.wait(0)
            sa_r, sb_r = o.restore_end(), r.wait(1)
            assert np.array_equal(sa_r, sb_r) and np.array_equal(sa_o, sb_o)
            p.check_claims(prev, "restore(k)")
            assert np.array_equal(o.release(prev), r.release(prev))
        p.check_claims(ids, "offload(k+1)", host=True)
        p.check_pool_state("interleaved", bytes_too=True)
        p.poison_free()
        prev = ids
    assert np.array_equal(o.restore(prev), r.restore(prev))
    p.check_pool_state("last restore")
    ev = p.check_events("interleaved")
    ok, why = V.validate(ev)
    assert ok, why
    p.close()


def test_two_open_offloads_run_ahead_of_a_restore():
    """rc.h split forms: up to two offloads may be open; each takes effect (reference drop, OFFLOADED) at its rc_wait(0),
    each restore at its _begin.  The bench schedule -- restore(k) in flight, offload(k+1) and offload(k+2) queued behind
    each other on the D2H side -- must equal the oracle making the synchronous calls in exactly that order; a third open
    offload is refused; rc_test never blocks."""
    wl = W.make_workload(0, n_claims=32, pool_blocks=2048)      # tiny geometry: claim 6 is PRED_FALSE, claim 3 has a fault
    p = Pair(wl, 1 << 30, chunk_blocks=37)                      # ~7 ragged chunks per wave
    o, r = p.o, p.r
    waves = W.plan_waves(wl, 1 << 30, max_claims_per_wave=8)
    assert len(waves) == 4
    top = wl.geom.pool_blocks

    def admit(wave):                                            # tables at the top of the pool, restores land at the bottom
        nonlocal top
        cl = [wl.claims[k] for k in wave.claim_idx]
        ids = [c.claim_id for c in cl]
        remap = np.zeros(wl.geom.pool_blocks, np.uint32)
        top -= wave.used_ids.size
        remap[wave.used_ids] = np.arange(top, top + wave.used_ids.size, dtype=np.uint32)
        p.set_fill(remap[wave.fill_ids], wave.fill_val)
        assert o.mark_used(remap[wave.used_ids]) == 0 and r.mark_used(remap[wave.used_ids]) == 0
        args = (ids, [c.P for c in cl], [c.N for c in cl], wave.bt_off, remap[wave.bt_ids])
        assert np.array_equal(o.accept(*args), r.accept(*args))
        assert np.array_equal(o.materialize(ids), r.materialize(ids))
        return ids

    ids = [admit(w) for w in waves]
    assert r.test(0) and r.test(1)                              # nothing in flight
    st_none = r.offload_begin([987654321])                      # nothing served: no operation is opened, statuses are final
    assert list(st_none) == [rc.ST_UNKNOWN_CLAIM] and list(o.offload([987654321])) == [rc.ST_UNKNOWN_CLAIM]
    r.offload_begin(ids[0])
    r.offload_begin(ids[1])
    rc3, _ = r._batch(r.L.rc_offload_begin, "rc_offload_begin", ids[2], check=False)
    assert rc3 == rc.ERR_BUSY                                   # a third open offload is refused and changes nothing
    assert list(r.wait(0)) == [rc.ST_UNKNOWN_CLAIM]             # the wait of the _begin that opened nothing: no library call
    assert np.array_equal(o.offload(ids[0]), r.wait(0))         # completes O0 only
    p.check_claims(ids[0], "O0", host=True)
    assert r.claim_info(ids[1][0])["state"] == 2                # O1 is open: still MATERIALIZED, blocks still referenced
    assert r.host_read(ids[1][0]) is None and r.host_store(ids[1][0], 0) is None   # RC_ERR_BUSY: its host copy is not complete yet
    for k in range(3):
        p.poison_free()
        fl = [(ids[k][1], rc.FAULT_BITFLIP, 12345 + k)] if k != 1 else [(ids[k][2], rc.FAULT_XFER_ERROR, 0)]
        fl += wl_faults(wl, ids[k])
        assert o.set_faults(fl) == 0 and r.set_faults(fl) == 0
        sa_r = o.restore(ids[k])                                # oracle: R(k), then O(k+1) where cuda completes it
        r.restore_begin(ids[k])
        if k + 2 < 4:
            r.offload_begin(ids[k + 2])                         # open now: O(k+1), O(k+2); R(k) in flight
        while not (r.test(0) and r.test(1)):
            pass
        assert np.array_equal(sa_r, r.wait(1))
        assert np.array_equal(o.offload(ids[k + 1]), r.wait(0))
        p.check_claims(ids[k], "R%d" % k)
        p.check_claims(ids[k + 1], "O%d" % (k + 1), host=True)
        p.check_pool_state("round %d" % k, bytes_too=True)
        assert np.array_equal(o.release(ids[k]), r.release(ids[k]))
    p.poison_free()
    assert np.array_equal(o.restore(ids[3]), r.restore(ids[3]))
    p.check_pool_state("last restore")
    back = [c for c in ids[3] if r.claim_info(c)["state"] == 4]
    r.offload_begin(back[:4])                                   # two open offloads completed by rc_sync, in _begin order
    r.offload_begin(back[4:])
    o.offload(back[:4]), o.offload(back[4:])
    r.sync()
    p.check_claims(back, "sync", host=True)
    p.check_pool_state("sync", bytes_too=False)
    ev = p.check_events("two open offloads")
    ok, why = V.validate(ev)
    assert ok, why
    s = r.stats()
    assert o.link_bytes() == (s["bytes_d2h"], s["bytes_h2d"])
    p.close()


def wl_faults(wl, ids):
    """the workload's own fault entries for the claims in ids"""
    want = set(ids)
    return [(c.claim_id,) + c.fault for c in wl.claims if c.fault and c.claim_id in want]


def test_edge_cases_fail_closed():
    """Empty batches, unknown / duplicate ids, bad tables, restore-after-use, host-store and
    free-block exhaustion: statuses and (absence of) events equal the oracle's."""
    wl = W.make_workload(0)
    g = wl.geom
    host = 70 * g.blk_bytes                                    # room for two claims only (28-32 blocks each)
    p = Pair(wl, host, chunk_blocks=7)
    o, r = p.o, p.r
    wave = W.plan_waves(wl, 1 << 30)[0]
    cl = wl.claims
    ids = [c.claim_id for c in cl]
    p.set_fill(wave.fill_ids, wave.fill_val)
    for x in (o, r):
        assert x.mark_used(wave.used_ids) == 0
        assert len(x.accept([], [], [], [0], [])) == 0 and len(x.offload([])) == 0 and len(x.restore([])) == 0
    # bad tables: out of range id, repeated id, unused block, wrong length, N > P, id 0, in-batch duplicate id
    t0 = wave.bt_ids[wave.bt_off[0]:wave.bt_off[1]].copy()
    free_blk = int(np.setdiff1d(np.arange(g.pool_blocks), wave.used_ids)[0]) if wave.used_ids.size < g.pool_blocks else None
    cases = []
    bad = t0.copy(); bad[3] = g.pool_blocks + 5; cases.append((ids[0], cl[0].P, 448, bad))
    bad = t0.copy(); bad[5] = bad[1]; cases.append((ids[0], cl[0].P, 448, bad))
    if free_blk is not None:
        bad = t0.copy(); bad[2] = free_blk; cases.append((ids[0], cl[0].P, 448, bad))
    cases.append((ids[0], cl[0].P, 448, t0[:-1]))
    cases.append((ids[0], cl[0].P, cl[0].P + 1, t0))
    cases.append((0, cl[0].P, 448, t0))
    cases.append((ids[0], cl[0].P, 448, t0))                   # valid
    cases.append((ids[0], cl[0].P, 448, t0))                   # duplicate of the previous, same batch
    off = np.cumsum([0] + [len(c[3]) for c in cases]).astype(np.uint32)
    args = ([c[0] for c in cases], [c[1] for c in cases], [c[2] for c in cases], off, np.concatenate([c[3] for c in cases]))
    sa, sb = o.accept(*args), r.accept(*args)
    assert np.array_equal(sa, sb) and list(sa[-2:]) == [0, 4]
    rest = list(range(1, len(cl)))
    args = ([ids[k] for k in rest], [cl[k].P for k in rest], [cl[k].N for k in rest],
            wave.bt_off[1:] - wave.bt_off[1], wave.bt_ids[wave.bt_off[1]:])
    assert np.array_equal(o.accept(*args), r.accept(*args))
    unknown = 0xDEADBEEF
    q = ids + [unknown, ids[0]]
    for fn in ("materialize", "offload", "restore"):           # offload: only the first two claims fit the host store
        sa, sb = getattr(o, fn)(q), getattr(r, fn)(q)
        assert np.array_equal(sa, sb), (fn, sa, sb)
        p.check_claims(ids, fn)
        p.check_pool_state(fn)
    assert np.array_equal(o.restore(q), r.restore(q))          # restore-after-use: BAD_STATE everywhere
    # free-block exhaustion at restore: offload two more, occupy the pool, restore both
    sa, sb = o.offload(ids[2:4]), r.offload(ids[2:4])
    assert np.array_equal(sa, sb) and list(sa) == [0, 0]
    used, _ = o.pool_state()
    free = np.nonzero(used == 0)[0].astype(np.uint32)
    keep = o.claim_info(ids[2])["nb"] + 3
    for x in (o, r):
        x.mark_used(free[keep:])
    sa, sb = o.restore(ids[2:4]), r.restore(ids[2:4])
    assert np.array_equal(sa, sb) and list(sa) == [0, 6]
    p.check_claims(ids, "exhaustion")
    p.check_pool_state("exhaustion")
    ev = p.check_events("edge")
    ok, why = V.validate(ev)
    assert ok, why
    p.close()


def test_determinism_repeated_runs():
    """The analogue of 131/131 valid sequences: repeated runs give byte-identical streams."""
    streams = []
    for _ in range(3):
        wl = W.make_workload(0)
        p = Pair(wl, 1 << 30, chunk_blocks=9)
        ev, _ = p.run_wave(W.plan_waves(wl, 1 << 30)[0])
        streams.append(ev.tobytes())
        p.close()
    assert streams[0] == streams[1] == streams[2]


def test_standalone_digest_matches_oracle():
    import torch
    wl = W.make_workload(0)
    g = wl.geom
    p = Pair(wl, 1 << 30, chunk_blocks=6)
    x = torch.randint(0, 256, (20 * g.blk_bytes,), dtype=torch.uint8, device="cuda")
    (d, e), ms = p.r.digest_blocks(x.data_ptr(), 20, both=True)
    xh = x.cpu().numpy()
    for which, got in ((0, d), (1, e)):
        want = [rco.block_digest(xh[i * g.blk_bytes:(i + 1) * g.blk_bytes], 2 * g.layers, which) for i in range(20)]
        assert [int(v) for v in got] == want
    p.close()


def test_host_store_fragmentation_ring_wrap_and_capacity():
    """Host-store extents split across free holes (space is granted by byte count, not contiguity), event
    ring wrap-around, RC_ERR_CAPACITY without side effects, release in every state."""
    wl = W.make_workload(0)
    g = wl.geom
    wave = W.plan_waves(wl, 1 << 30)[0]
    cl = wl.claims
    ids = [c.claim_id for c in cl]
    ok = [k for k in range(len(cl)) if k != 6]
    nb = {c.claim_id: (c.M + g.block_size - 1) // g.block_size for c in cl}
    host_blocks = sum(nb[ids[k]] for k in ok[:4]) + 3                     # room for four claims and a bit
    p = Pair(wl, host_blocks * g.blk_bytes, chunk_blocks=13, max_events=24)
    o, r = p.o, p.r
    p.set_fill(wave.fill_ids, wave.fill_val)
    for x in (o, r):
        assert x.mark_used(wave.used_ids) == 0
    args = (ids, [c.P for c in cl], [c.N for c in cl], wave.bt_off, wave.bt_ids)
    assert np.array_equal(o.accept(*args), r.accept(*args))
    assert np.array_equal(o.materialize(ids), r.materialize(ids))
    ea = p.check_events("drain 1")                                        # 8 + 7 events: ring of 24 wraps below
    a4 = [ids[k] for k in ok[:4]]
    assert np.array_equal(o.offload(a4), r.offload(a4))
    # free the 1st and 3rd slots, then offload a claim that only fits split across the two holes + tail
    p.poison_free()
    assert np.array_equal(o.restore([a4[0], a4[2]]), r.restore([a4[0], a4[2]]))
    p.check_events("drain 2")
    big = [ids[k] for k in ok[4:6]]
    sa, sb = o.offload(big), r.offload(big)
    assert np.array_equal(sa, sb) and sa[0] == 0
    p.check_claims(ids, "fragmented offload", host=True)
    p.poison_free()
    q = [a4[1], a4[3]] + big
    assert np.array_equal(o.restore(q), r.restore(q))
    p.check_claims(ids, "fragmented restore")
    p.check_pool_state("fragmented restore")
    ev = p.check_events("drain 3")
    assert int(ev["seq"][-1]) > 24                                        # the ring wrapped and stayed gap-free
    # event capacity: with 13 records pending, 3 more restores (up to 12 records) do not fit a ring of 24:
    # RC_ERR_CAPACITY, and nothing changes
    more = [ids[k] for k in ok]
    sa, sb = o.offload(more), r.offload(more)
    assert np.array_equal(sa, sb) and list(sa).count(0) == 4
    live = [c for c, s_ in zip(more, sa) if s_ == 0]
    for _ in range(3):
        assert np.array_equal(o.restore(live[:1]), r.restore(live[:1]))
        assert np.array_equal(o.offload(live[:1]), r.offload(live[:1]))
    rcode, st = r.restore(live[1:], check=False)
    assert rcode == rc.ERR_CAPACITY
    assert all(r.claim_info(c)["state"] == 3 for c in live)
    p.check_pool_state("capacity error", bytes_too=False)
    p.check_events("drain after capacity error")
    more = live
    # release in every state: ACCEPTED (claim 6), OFFLOADED, then restored ones
    assert np.array_equal(o.restore(more[:3]), r.restore(more[:3]))
    p.check_events("drain 4")
    assert np.array_equal(o.release(ids + [ids[0]]), r.release(ids + [ids[0]]))
    p.check_pool_state("release all", bytes_too=False)
    assert r.stats()["host_used_bytes"] == 0 == o.stats()["host_used"]
    p.close()


def test_bitflip_positions_across_chunk_boundaries():
    """The injected corruption lands in the first / last byte of the claim and on both sides of a staging
    chunk boundary; LOAD_FAILED.aux is the block that holds the flipped byte (affected-block evidence)."""
    wl = W.make_workload(0)
    g = wl.geom
    wave = W.plan_waves(wl, 1 << 30)[0]
    cl = wl.claims
    ids = [c.claim_id for c in cl]
    blk = g.blk_bytes
    nb0 = (cl[0].M + g.block_size - 1) // g.block_size
    params = [0, nb0 * blk - 1, 7 * blk - 1, 7 * blk, 3 * blk + 12345]      # chunk = 7 blocks
    for prm, k in zip(params, (0, 0, 0, 0, 1)):
        p = Pair(wl, 1 << 30, chunk_blocks=7)
        ev, st = p.run_wave(wave, faults=[(ids[k], W.FK_BITFLIP, prm)])
        lf = [e for e in ev if int(e["code"]) == 5]
        assert len(lf) == 1 and int(lf[0]["claim_id"]) == ids[k] and int(lf[0]["aux"]) == prm // blk
        assert st[k] == rc.ST_RESTORE_FAILED and st.count(rc.ST_RESTORE_FAILED) == 1
        p.close()


# ---- NEXT-2: content-addressed host store (dedup) ------------------------------------------------------
@pytest.mark.parametrize("mover", [rc.MOVER_TMA, rc.MOVER_LDG])
@pytest.mark.parametrize("chunk_blocks", [9, 64])
def test_dedup_shared_tiny_full_parity(mover, chunk_blocks):
    """Shared prefixes + identical content in different blocks: one held copy and one link transfer per
    distinct block, everything else (bytes, digests, chains, events, allocation) as without dedup."""
    wl, wave, copies = make_shared_tiny()
    ids = [c.claim_id for c in wl.claims]
    p = Pair(wl, 1 << 30, chunk_blocks=chunk_blocks, mover=mover, dedup=True, copies=copies)
    g = wl.geom
    wave.faults = [(ids[0], W.FK_BITFLIP, 5 * g.blk_bytes + 17), (ids[3], W.FK_XFER_ERROR, 0)]
    ev, st = p.run_wave(wave, restore_batches=[ids[:3], ids[3:]])
    assert st == [8, 0, 0, 8, 0, 0]                              # the shared block's corruption stays on claim 0
    s = p.r.stats()
    total = sum((c.M + g.block_size - 1) // g.block_size for c in wl.claims) * g.blk_bytes
    assert s["bytes_d2h"] < total - 20 * g.blk_bytes and s["bytes_h2d"] < total
    ok, why = V.validate(ev)
    assert ok, why
    p.close()


def test_dedup_config2_shared_prefixes_reduced():
    wl = W.make_workload(2, n_claims=4, pool_blocks=1300)
    host = 6 << 30
    p = Pair(wl, host, chunk_blocks=50, dedup=True)
    for wave in W.plan_waves(wl, host):
        ids = [wl.claims[k].claim_id for k in wave.claim_idx]
        ev, _ = p.run_wave(wave, restore_batches=[ids[i:i + 2] for i in range(0, len(ids), 2)])
        ok, why = V.validate(ev)
        assert ok, why
    p.close()


def test_dedup_overlapped_begin_wait_matches_synchronous_order():
    """restore(k) in flight while offload(k+1) dedups against the store: the restore holds its references until
    rc_wait(1), so blocks of k that reappear in k+1 are not copied again; equal to the oracle making the same split calls."""
    wl, wave, copies = make_shared_tiny()
    ids = [c.claim_id for c in wl.claims]
    p = Pair(wl, 1 << 30, chunk_blocks=11, dedup=True, copies=copies)
    o, r = p.o, p.r
    p.set_fill(wave.fill_ids, wave.fill_val)
    for x in (o, r):
        assert x.mark_used(wave.used_ids) == 0
    args = (ids, [c.P for c in wl.claims], [c.N for c in wl.claims], wave.bt_off, wave.bt_ids)
    assert np.array_equal(o.accept(*args), r.accept(*args))
    assert np.array_equal(o.materialize(ids), r.materialize(ids))
    a, b = ids[:3], ids[3:]
    assert np.array_equal(o.offload(a), r.offload(a))
    p.poison_free()
    o.restore_begin(a)
    r.restore_begin(a)
    r.offload_begin(b)                       # the store is looked up now: a's blocks are still held by the restore in flight
    sa_o, sb_o = o.offload(b), r.wait(0)
    sa_r, sb_r = o.restore_end(), r.wait(1)
    assert np.array_equal(sa_r, sb_r) and np.array_equal(sa_o, sb_o)
    p.check_claims(ids, "overlap", host=True)
    p.check_pool_state("overlap")
    s = r.stats()
    assert o.link_bytes() == (s["bytes_d2h"], s["bytes_h2d"]) and o.stats()["host_used"] == s["host_used_bytes"]
    p.poison_free()
    assert np.array_equal(o.restore(b), r.restore(b))
    p.check_pool_state("final")
    p.check_events("overlap")
    assert np.array_equal(o.release(ids), r.release(ids))
    assert r.stats()["host_used_bytes"] == 0
    p.close()


# ---- NEXT-3: multi-claim reuse requests, demotion / expiry ------------------------------------------------
@pytest.mark.parametrize("dedup", [False, True])
def test_requests_and_failure_policies_parity(dedup):
    """One reuse request over several claims: refusal names exactly the failed subset;
    demotion / expiry as the claim's outcome of a failed restoration.  Events, statuses, states and
    pool state equal the oracle's; overlapped begin/wait form included."""
    wl = W.make_workload(0)
    wave = W.plan_waves(wl, 1 << 30)[0]
    cl = wl.claims
    ids = [c.claim_id for c in cl]
    p = Pair(wl, 1 << 30, chunk_blocks=10, dedup=dedup)
    o, r = p.o, p.r
    p.set_fill(wave.fill_ids, wave.fill_val)
    for x in (o, r):
        assert x.mark_used(wave.used_ids) == 0
    args = (ids, [c.P for c in cl], [c.N for c in cl], wave.bt_off, wave.bt_ids)
    assert np.array_equal(o.accept(*args), r.accept(*args))
    assert np.array_equal(o.materialize(ids), r.materialize(ids))
    ok = [ids[k] for k in range(8) if k != 6]
    assert np.array_equal(o.offload(ok), r.offload(ok))
    p.poison_free()
    for x in (o, r):
        assert x.set_policy([ok[0], ok[1]], [1, 2]) == 0
        assert x.set_policy([0xBAD], [1]) != 0 and x.set_policy([ok[2]], [7]) != 0
        assert x.set_faults([(ok[0], W.FK_XFER_ERROR, 0), (ok[1], W.FK_BITFLIP, 3), (ok[2], W.FK_XFER_ERROR, 0),
                             (ok[4], W.FK_BITFLIP, 77777)]) == 0
    req = 0x5151
    q = ok[:5] + [ids[6], 0xFEED]                               # + a PRED_FALSE claim and an unknown id
    sa, sb = o.restore_request(req, q), r.restore_request(req, q)
    assert np.array_equal(sa, sb) and list(sa) == [8, 8, 8, 0, 8, 3, 2]
    p.check_claims(ids, "request")
    p.check_pool_state("request")
    ev = p.check_events("request")
    grp = [e for e in ev if int(e["code"]) == 8]
    assert [int(e["claim_id"]) for e in grp] == [ok[2], ok[4]] and all(int(e["aux"]) == (rc.REQ_FLAG | 2) for e in grp)
    ok_, why = V.validate(ev)
    assert ok_, why
    # second request, overlapped form, no failure -> no refusal record
    sa = o.restore_request(req + 1, ok[5:])
    r.restore_request_begin(req + 1, ok[5:])
    sb = r.wait(1)
    assert np.array_equal(sa, sb) and not sa.any()
    ev2 = p.check_events("request 2")
    assert 8 not in [int(e["code"]) for e in ev2]
    assert np.array_equal(o.restore(ok), r.restore(ok))         # all terminal or resident: BAD_STATE everywhere
    rcode, _ = r.restore_request(0, ok, check=False)
    assert rcode == rc.ERR_INVALID
    p.close()


@pytest.mark.parametrize("mover", [rc.MOVER_TMA, rc.MOVER_LDG])
def test_direct_offload_into_mapped_pinned_store(mover):
    """NEXT-4 (first half): the gather kernel's stores cross the link themselves; every observable unchanged."""
    wl = W.make_workload(0)
    p = Pair(wl, 1 << 30, chunk_blocks=9, mover=mover, direct_offload=True)
    ev, st = p.run_wave(W.plan_waves(wl, 1 << 30)[0])
    assert st[3] == rc.ST_RESTORE_FAILED and V.validate(ev)[0]
    p.close()


# ---- NEXT-4: layer-major streaming order (rc_config.layer_major; DESIGN R28) ----------------------------------------------
@pytest.mark.parametrize("mover", [rc.MOVER_LDG, rc.MOVER_TMA])
@pytest.mark.parametrize("kind", [W.FK_BITFLIP, W.FK_XFER_ERROR])
@pytest.mark.parametrize("chunk_blocks", [5, 64, 300])
def test_layer_major_tiny_full_parity(mover, kind, chunk_blocks):
    """Host copy [g][block][page], staging chunks [g][item][page]: host bytes, digests, chains, allocation, pool bytes and
    events against the oracle in the same mode, with chunks that cut claims (5), hold two claims (64) or the whole wave."""
    wl = W.make_workload(0)
    p = Pair(wl, 1 << 30, chunk_blocks=chunk_blocks, mover=mover, layer_major=True)
    wave = W.plan_waves(wl, 1 << 30)[0]
    faults = [(cid, kind, prm) for cid, _, prm in wave.faults]
    ev, st_r = p.run_wave(wave, faults=faults)
    assert V.validate(ev)[0]
    assert names(ev, wl.claims[3].claim_id) == GOLD["failure_path"] and st_r[3] == rc.ST_RESTORE_FAILED
    assert p.r.host_store(wl.claims[0].claim_id, 0) is None          # no contiguous block in this layout
    p.close()


def test_layer_major_fragmented_host_store_and_interleaved_waves():
    """Claims whose host copy is split over several extents of the store (the plane runs straddle the pieces), bit flips
    on both sides of plane and chunk boundaries, restore(k) in flight with two offloads open."""
    wl = W.make_workload(4, n_claims=24, pool_blocks=3072, scale=64)
    host = 3 << 30
    p = Pair(wl, host, chunk_blocks=64, layer_major=True)
    o, r = p.o, p.r
    waves = W.plan_waves(wl, host, max_claims_per_wave=8)
    blk, page = wl.geom.blk_bytes, wl.geom.page_bytes

    def admit(wave):
        cl = [wl.claims[k] for k in wave.claim_idx]
        ids = [c.claim_id for c in cl]
        used, _ = o.pool_state()
        free = np.nonzero(used == 0)[0].astype(np.uint32)
        remap = np.zeros(wl.geom.pool_blocks, np.uint32)
        remap[wave.used_ids] = free[: wave.used_ids.size]
        p.set_fill(remap[wave.fill_ids], wave.fill_val)
        assert o.mark_used(remap[wave.used_ids]) == 0 and r.mark_used(remap[wave.used_ids]) == 0
        args = (ids, [c.P for c in cl], [c.N for c in cl], wave.bt_off, remap[wave.bt_ids])
        assert np.array_equal(o.accept(*args), r.accept(*args))
        assert np.array_equal(o.materialize(ids), r.materialize(ids))
        return ids

    # fragment the host store: offload wave 0 claim by claim, release every second claim
    ids0 = admit(waves[0])
    for c in ids0:
        assert np.array_equal(o.offload([c]), r.offload([c]))
    assert np.array_equal(o.release(ids0[::2]), r.release(ids0[::2]))
    ids1 = admit(waves[1])
    assert np.array_equal(o.offload(ids1), r.offload(ids1))            # lands in the holes: split extents
    p.check_claims(ids1, "offload into a fragmented store", host=True)
    nb, nb2 = r.claim_info(ids1[0])["nb"], r.claim_info(ids1[2])["nb"]
    flips = [(ids1[0], rc.FAULT_BITFLIP, 2 * nb * page - 1), (ids1[1], rc.FAULT_BITFLIP, 0),
             (ids1[2], rc.FAULT_BITFLIP, nb2 * blk - 1)]
    p.poison_free()
    assert o.set_faults(flips) == 0 and r.set_faults(flips) == 0
    ids2 = admit(waves[2])
    o.restore_begin(ids1)
    r.restore_begin(ids1)
    r.offload_begin(ids2[:4])
    r.offload_begin(ids2[4:])
    sa = [o.offload(ids2[:4]), o.offload(ids2[4:])]
    assert np.array_equal(sa[0], r.wait(0)) and np.array_equal(sa[1], r.wait(0))
    sa_r, sb_r = o.restore_end(), r.wait(1)
    assert np.array_equal(sa_r, sb_r) and list(sb_r[:3]) == [8, 8, 8]
    p.check_claims(ids1 + ids2, "interleaved", host=False)
    p.check_claims(ids2, "offloaded", host=True)
    p.check_pool_state("interleaved", bytes_too=True)
    ev = p.check_events("layer-major")
    assert V.validate(ev)[0]
    bad = [int(e["aux"]) for e in ev if int(e["code"]) == 5]
    assert bad == [nb - 1, 0, nb2 - 1]            # the block that the layer-major layout puts at each flipped byte
    p.close()


def test_large_batch_multi_tile_scans():
    """3000 claims in one batch on a 98304-block pool: every single-CTA scan (offsets, restore plan, allocation,
    event emission) runs over several tiles with carries; sub-batched restores hit NO_FREE_BLOCKS prefixes."""
    wl = W.make_workload(0, n_claims=3000, pool_blocks=98304)
    rng = np.random.default_rng(11)
    for k in range(0, 3000, 97):
        wl.claims[k].fault = (W.FK_XFER_ERROR, 0) if (k // 97) % 2 else (W.FK_BITFLIP, int(rng.integers(0, 1 << 31)))
    for k in range(5, 3000, 211):
        wl.claims[k].M = int(rng.integers(0, 448))          # under-materialized: PRED_FALSE
        wl.claims[k].fault = None
    host = 2 << 30
    p = Pair(wl, host, chunk_blocks=4096, max_events=1 << 16)
    waves = W.plan_waves(wl, host)
    assert len(waves) == 1 and len(waves[0].claim_idx) == 3000
    ids = [c.claim_id for c in wl.claims]
    ev, st = p.run_wave(waves[0], restore_batches=[ids[:1500], ids[1500:]], check_bytes=False)
    assert st.count(rc.ST_RESTORE_FAILED) == sum(1 for c in wl.claims if c.fault)
    assert st.count(rc.ST_BAD_STATE) == sum(1 for c in wl.claims if c.M < c.N)
    ok, why = V.validate(ev)
    assert ok, why
    # occupy most of the pool, then restore a batch that only partly fits: prefix grant across scan tiles
    o, r = p.o, p.r
    ok_ids = [c.claim_id for c in wl.claims if c.M >= c.N][:2000]
    p.set_fill(waves[0].fill_ids, waves[0].fill_val)
    for x in (o, r):
        assert x.mark_used(waves[0].used_ids) == 0
    args = (ids, [c.P for c in wl.claims], [c.N for c in wl.claims], waves[0].bt_off, waves[0].bt_ids)
    assert np.array_equal(o.accept(*args), r.accept(*args))
    assert np.array_equal(o.materialize(ids), r.materialize(ids))
    assert np.array_equal(o.offload(ok_ids), r.offload(ok_ids))
    used, _ = o.pool_state()
    free = np.nonzero(used == 0)[0].astype(np.uint32)
    for x in (o, r):
        x.mark_used(free[40000:])                             # leave 40000 free blocks: about 1300 claims fit
    sa, sb = o.restore(ok_ids), r.restore(ok_ids)
    assert np.array_equal(sa, sb) and 0 in sa and 6 in sa
    first6 = list(sa).index(6)
    assert all(s == 6 for s in sa[first6:]) and first6 > 1024     # the grant boundary lies beyond the first scan tile
    p.check_pool_state("partial grant", bytes_too=False)
    p.check_events("partial grant")
    p.close()


def test_predicate_on_random_non_monotone_fill():
    """500 claims whose fill vectors are NOT 'full blocks, one partial, zeros': holes followed by full blocks, a zero
    first block, fill above the token count of a short last block.  M is the LEADING run of materialized tokens
    (P:L25 'leading-prefix-at-least-448'): k_pred must agree with the oracle, and both with the token-level definition
    restated here; a predicate that summed fills would differ on most of these claims."""
    wl = W.make_workload(0, n_claims=500, pool_blocks=16384)
    g = wl.geom
    BS = g.block_size
    wave = W.plan_waves(wl, 1 << 40)[0]
    rng = np.random.default_rng(23)
    fill = np.zeros(g.pool_blocks, np.uint8)
    want_M, differs = [], 0
    for k, c in enumerate(wl.claims):
        c.fault = None
        tab = wave.bt_ids[wave.bt_off[k]:wave.bt_off[k + 1]]
        nt = len(tab)
        f = rng.integers(0, BS + 1, nt)                                    # arbitrary fills everywhere ...
        kind = k % 5
        lead = nt if kind == 0 else (0 if kind == 1 else int(rng.integers(max(0, nt - 6), nt + 1)))
        f[:lead] = BS                                                      # ... behind `lead` complete blocks
        if kind == 2 and lead < nt:
            f[lead] = int(rng.integers(0, BS))                             # the hole
            f[lead + 1:] = BS                                              # and full blocks after it
        if kind == 3:
            f[-1] = BS                                                     # fill above the tokens of the short last block
        fill[tab] = f
        M = next((t for t in range(c.P) if not (t % BS) < f[t // BS]), c.P)
        want_M.append(M)
        differs += int(sum(min(int(f[i]), min(BS, c.P - i * BS)) for i in range(nt)) != M)
    assert differs > 200
    p = Pair(wl, 1 << 32, chunk_blocks=512)
    o, r = p.o, p.r
    p.set_fill(np.arange(g.pool_blocks), fill)
    ids = [c.claim_id for c in wl.claims]
    for x in (o, r):
        assert x.mark_used(wave.used_ids) == 0
    args = (ids, [c.P for c in wl.claims], [c.N for c in wl.claims], wave.bt_off, wave.bt_ids)
    assert np.array_equal(o.accept(*args), r.accept(*args))
    sa, sb = o.materialize(ids), r.materialize(ids)
    assert np.array_equal(sa, sb)
    assert [int(s) for s in sa] == [0 if M >= c.N else 1 for M, c in zip(want_M, wl.claims)]
    assert 100 < int((sa == 0).sum()) < 400
    for c, M, s in zip(wl.claims, want_M, sa):
        if s == 0:
            assert r.claim_info(c.claim_id)["M"] == M == o.claim_info(c.claim_id)["M"]
    p.check_claims(ids, "materialize", digests=False)
    sa, sb = o.offload(ids), r.offload(ids)
    assert np.array_equal(sa, sb)
    p.check_claims(ids, "offload", host=True)
    p.poison_free()
    assert np.array_equal(o.restore(ids), r.restore(ids))
    p.check_claims(ids, "restore")
    p.check_pool_state("restore")                                          # fill of restored blocks = min(BS, M - i*BS)
    ev = p.check_events("random fill")
    assert [int(e["aux"]) for e in ev if int(e["code"]) == 2] == [M for M, s in zip(want_M, sa) if s != 3 and M >= 448]
    assert V.validate(ev)[0]
    p.close()


def test_call_level_errors_change_nothing():
    """rc.h: a negative return emits no event and changes no claim: RC_ERR_CAPACITY of rc_accept in a later
    run of a batch with a duplicate id, RC_ERR_CAPACITY of rc_offload after digests were recorded by an earlier cycle,
    RC_ERR_BUSY of rc_measure_link while the pinned store holds claim bytes."""
    import torch
    wl = W.make_workload(0)
    g = wl.geom
    wave = W.plan_waves(wl, 1 << 30)[0]
    cl = wl.claims
    pool = W.pool_torch(g, torch.device("cuda:0"))
    fill = torch.zeros(g.pool_blocks, dtype=torch.uint8, device="cuda:0")
    fill[torch.from_numpy(wave.fill_ids.astype(np.int64)).cuda()] = torch.from_numpy(wave.fill_val).cuda()
    torch.cuda.synchronize()
    r = rc.RC(g.layers, g.kv_heads, g.head_dim, g.elem_bytes, g.block_size, g.pool_blocks, pool, fill, 1 << 30,
              staging_chunk_bytes=16 * g.blk_bytes, max_table_entries=100)
    assert r.mark_used(wave.used_ids) == 0
    tabs = [wave.bt_ids[wave.bt_off[k]:wave.bt_off[k + 1]] for k in range(4)]
    ids = [c.claim_id for c in cl[:4]]

    def batch(ks):
        off = np.cumsum([0] + [len(tabs[k]) for k in ks]).astype(np.uint32)
        return ([ids[k] for k in ks], [cl[k].P for k in ks], [448] * len(ks), off, np.concatenate([tabs[k] for k in ks]))
    # claims 0, 0 (duplicate id: second run), 1, 2: 4 x ~30 table entries do not fit 100 -> nothing is accepted
    rcode, st = r.accept(*batch([0, 0, 1, 2]), check=False)
    assert rcode == rc.ERR_CAPACITY and len(r.outcomes()) == 0 and all(r.claim_info(c) is None for c in ids)
    _, ref = r.pool_state()
    assert not ref.any()
    assert list(r.accept(*batch([0, 0, 1]))) == [0, 4, 0]                 # the same duplicate, now within capacity
    assert not r.materialize(ids[:2]).any() and not r.offload(ids[:2]).any()
    with pytest.raises(rc.RcError) as ei:
        r.measure_link(1 << 20, 0, reps=1)                                 # would write over the claims' host copies
    assert ei.value.code == rc.ERR_BUSY
    hb = r.host_read(ids[0]).copy()
    assert not r.restore(ids[:2]).any()
    d0 = r.claim_digests(ids[0]).copy()
    info0 = r.claim_info(ids[0])
    # second cycle: the new digest extent is taken before the old one is given back; 2 x ~30 held + ~30 + ~30 new > 100
    rcode, st = r.offload(ids[:2], check=False)
    assert rcode == rc.ERR_CAPACITY
    assert r.claim_info(ids[0]) == info0 and np.array_equal(r.claim_digests(ids[0]), d0)     # state and digests intact
    assert r.stats()["host_used_bytes"] == 0 and len(r.outcomes()) == 10                    # 2 x (A, M, O, RR, R): no new event
    assert list(r.offload(ids[:1])) == [0]                                                  # one claim still fits
    assert np.array_equal(r.host_read(ids[0]), hb)
    r.close()


# ---- split forms under random interleavings -------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_split_forms_random_interleavings(seed):
    """Random legal sequences of admit / rc_offload_begin (up to two open) / rc_wait(0) / rc_restore_begin / rc_wait(1) /
    rc_release / poison, with other claims' metadata calls between a _begin and its rc_wait.  The oracle makes the calls rc.h
    says they are equal to: an offload at its rc_wait(0), a restore as rco_restore_begin at its _begin and rco_restore_end at
    its rc_wait(1).  Statuses, claim records, digests, host bytes, allocation and -- whenever nothing is in flight -- pool
    bytes are compared on the way, the whole event stream at the end.  The pool is small enough for NO_FREE_BLOCKS to occur;
    the host store is ample (an offload's host-space grant is taken at _begin: rc.h)."""
    rng = np.random.default_rng(1000 + seed)
    wl = W.make_workload(0, n_claims=48, pool_blocks=160)        # ~5 claims fit: NO_FREE_BLOCKS is common
    g = wl.geom
    p = Pair(wl, 1 << 30, chunk_blocks=41)
    o, r = p.o, p.r
    todo = list(range(len(wl.claims)))
    resident, offloaded, back = [], [], []                     # claim ids by where they are (idle claims only)
    open_q, in_restore = [], None
    n_busy_status = n_nofree = 0

    def admit(k):
        c = wl.claims[k]
        nt = -(-c.P // g.block_size)
        used, _ = o.pool_state()
        free = np.nonzero(used == 0)[0].astype(np.uint32)
        if free.size < nt:
            return False
        tab = rng.choice(free[free.size // 2:] if free.size // 2 >= nt else free, nt, replace=False).astype(np.uint32)
        fv = np.array([min(g.block_size, max(0, c.M - i * g.block_size)) for i in range(nt)], np.uint8)
        p.set_fill(tab, fv)
        assert o.mark_used(tab) == 0 and r.mark_used(tab) == 0
        args = ([c.claim_id], [c.P], [c.N], [0, nt], tab)
        assert np.array_equal(o.accept(*args), r.accept(*args))
        sa, sb = o.materialize([c.claim_id]), r.materialize([c.claim_id])
        assert np.array_equal(sa, sb)
        if sa[0] == 0:
            resident.append(c.claim_id)
        else:                                                  # PRED_FALSE: give the blocks back
            assert np.array_equal(o.release([c.claim_id]), r.release([c.claim_id]))
            assert o.mark_free(tab) == 0 and r.mark_free(tab) == 0
        return True

    def pick(lst, lo=1, hi=6):
        n = int(rng.integers(lo, min(hi, len(lst)) + 1))
        ids = [lst.pop(int(rng.integers(0, len(lst)))) for _ in range(n)]
        return ids

    for step in range(260):
        acts = []
        if todo:
            acts.append("admit")
        if resident and len(open_q) < 2:
            acts += ["obegin"] * 2
        if open_q:
            acts += ["owait"] * 2
        if offloaded and in_restore is None:
            acts += ["rbegin"] * 2
        if in_restore is not None:
            acts.append("rwait")
        if back:
            acts.append("release")
        acts.append("poison")
        a = acts[int(rng.integers(0, len(acts)))]
        if a == "admit":
            if not admit(todo[0]):
                continue
            todo.pop(0)
        elif a == "obegin":
            ids = pick(resident)
            extra = []
            if open_q and rng.random() < 0.3:                  # a claim of an open offload answers BAD_STATE, no effect
                extra = [open_q[0][0][0]]
            st = r.offload_begin(ids + extra)
            if extra:
                assert st[-1] == rc.ST_BAD_STATE
                n_busy_status += 1
            open_q.append((ids, extra))
        elif a == "owait":
            ids, extra = open_q.pop(0)
            sb = r.wait(0)
            sa = o.offload(ids)
            assert np.array_equal(sa, sb[: len(ids)]) and not sa.any()
            p.check_claims(ids, "offload at rc_wait(0)", host=True)
            offloaded += ids
        elif a == "rbegin":
            ids = pick(offloaded)
            fl = []
            for c in ids:
                u = rng.random()
                if u < 0.15:
                    fl.append((c, rc.FAULT_BITFLIP, int(rng.integers(0, 1 << 31))))
                elif u < 0.25:
                    fl.append((c, rc.FAULT_XFER_ERROR, 0))
            assert o.set_faults(fl) == 0 and r.set_faults(fl) == 0
            sa, sb = o.restore_begin(ids), r.restore_begin(ids)
            assert np.array_equal(sa, sb), (sa, sb)            # -1 for served claims, final for the others (NO_FREE_BLOCKS)
            in_restore = ids
        elif a == "rwait":
            sa, sb = o.restore_end(), r.wait(1)
            assert np.array_equal(sa, sb), (sa, sb)
            p.check_claims(in_restore, "restore at rc_wait(1)")
            for c, s in zip(in_restore, sa):
                if s == 0:
                    back.append(c)
                elif s == rc.ST_NO_FREE_BLOCKS:
                    offloaded.append(c)
                    n_nofree += 1
            in_restore = None
        elif a == "release":
            ids = pick(back, 1, 4)
            assert np.array_equal(o.release(ids), r.release(ids))
        else:
            p.poison_free()
        if not open_q and in_restore is None and step % 7 == 0:
            p.check_pool_state("step %d" % step, bytes_too=True)
    while open_q:
        ids, extra = open_q.pop(0)
        assert np.array_equal(o.offload(ids), r.wait(0)[: len(ids)])
    if in_restore is not None:
        assert np.array_equal(o.restore_end(), r.wait(1))
    p.check_pool_state("end", bytes_too=True)
    ev = p.check_events("random interleavings")
    ok, why = V.validate(ev)
    assert ok, why
    assert len(ev) > 100 and n_nofree > 0 and n_busy_status > 0      # the refusals did occur
    s = r.stats()
    assert o.link_bytes() == (s["bytes_d2h"], s["bytes_h2d"]) and o.stats()["host_used"] == s["host_used_bytes"]
    p.close()


def test_set_fill_from_host_arrays():
    """rc_set_fill writes exactly the named entries of the caller's fill vector and refuses bad input without writing."""
    wl = W.make_workload(0)
    p = Pair(wl, 1 << 30)
    rng = np.random.default_rng(3)
    ids = rng.choice(wl.geom.pool_blocks, 100, replace=False).astype(np.uint32)
    vals = rng.integers(0, wl.geom.block_size + 1, 100).astype(np.uint8)
    want = p.fill_t.cpu().numpy().copy()
    want[ids] = vals
    p.r.set_fill(ids, vals)
    assert np.array_equal(p.fill_t.cpu().numpy(), want)
    for bad_ids, bad_vals in ((np.array([wl.geom.pool_blocks], np.uint32), np.array([1], np.uint8)),
                              (np.array([0], np.uint32), np.array([wl.geom.block_size + 1], np.uint8))):
        with pytest.raises(rc.RcError):
            p.r.set_fill(bad_ids, bad_vals)
    assert np.array_equal(p.fill_t.cpu().numpy(), want)
    p.r.set_fill(np.zeros(0, np.uint32), np.zeros(0, np.uint8))
    p.close()


@pytest.mark.parametrize("mode", ["plain", "dedup", "direct", "layer_major", "ldg"])
def test_checked_mode_finds_no_out_of_range_work_item(mode, monkeypatch):
    """RC_CHECK=1 (compute-sanitizer is closed on this pool): k_check_items validates the work items of every mover launch --
    pool block, work position, staged block -- and rc_wait refuses to complete an operation whose flag is set.  The Tiny
    wave with ragged chunks runs clean in every mover mode, and results do not change."""
    monkeypatch.setenv("RC_CHECK", "1")
    wl, wave = W.make_workload(0), None
    kw = dict(dedup=mode == "dedup", direct_offload=mode == "direct", layer_major=mode == "layer_major",
              mover=rc.MOVER_LDG if mode == "ldg" else rc.MOVER_AUTO)
    p = Pair(wl, 1 << 30, chunk_blocks=7, **kw)
    wave = W.plan_waves(wl, 1 << 30)[0]
    ev, st_r = p.run_wave(wave)
    assert V.validate(ev)[0] and st_r.count(rc.ST_RESTORE_FAILED) == 1
    assert p.r.stats()["kernel_launches"] > 0
    p.close()
