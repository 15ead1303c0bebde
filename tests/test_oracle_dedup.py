"""NEXT-2 pins: the content-addressed host store of the oracle (dedup mode) against what the definition fixes,
computed here independently with hashlib over the claim-logical bytes: one held copy and one link transfer
per distinct block content, unchanged claim-logical bytes / events / round trip, target-only attribution when
the corrupted block is shared."""
import hashlib

import numpy as np

from oracle import rco, validator as V
from paper_2606_01387_b200 import workloads as W
from shared_tiny import make_shared_tiny


def build(dedup, host=1 << 40):
    wl, wave, copies = make_shared_tiny()
    g = wl.geom
    pool = W.pool_host(g)
    view = pool.reshape(2 * g.layers, g.pool_blocks, g.page_bytes)
    for src, dst in copies:
        view[:, dst, :] = view[:, src, :]
    fill = np.zeros(g.pool_blocks, np.uint8)
    fill[wave.fill_ids] = wave.fill_val
    o = rco.Oracle(g.layers, g.kv_heads, g.head_dim, g.elem_bytes, g.block_size, g.pool_blocks, pool, fill, host)
    assert o.set_dedup(dedup) == 0
    o.mark_used(wave.used_ids)
    ids = [c.claim_id for c in wl.claims]
    assert not o.accept(ids, [c.P for c in wl.claims], [c.N for c in wl.claims], wave.bt_off, wave.bt_ids).any()
    assert not o.materialize(ids).any()
    return o, wl, wave, view, ids


def block_keys(view, table):
    return [hashlib.sha256(view[:, b, :].tobytes()).digest() for b in table]


def test_dedup_store_holds_and_moves_each_distinct_block_once():
    o, wl, wave, view, ids = build(True)
    g = wl.geom
    p, _, _, view_p, _ = build(False)
    keys = {cid: block_keys(view, wave.bt_ids[wave.bt_off[k]:wave.bt_off[k + 1]]) for k, cid in enumerate(ids)}
    logical = {cid: o.claim_blocks(cid) for cid in ids}
    before = {cid: view[:, logical[cid], :].transpose(1, 0, 2).copy() for cid in ids}
    assert not o.offload(ids[:4]).any() and not p.offload(ids[:4]).any()
    distinct = set(k for cid in ids[:4] for k in keys[cid])
    total = sum(len(keys[cid]) for cid in ids[:4])
    assert len(distinct) < total - 20                                          # the inputs really share
    assert o.stats()["host_used"] == len(distinct) * g.blk_bytes               # one held copy per content
    assert o.link_bytes() == (len(distinct) * g.blk_bytes, 0)                  # ... and one D2H transfer
    assert p.stats()["host_used"] == total * g.blk_bytes == p.link_bytes()[0]
    for cid in ids[:4]:                                                        # claim-logical bytes unchanged
        assert np.array_equal(o.host_read(cid), p.host_read(cid))
        assert np.array_equal(o.host_read(cid), before[cid].reshape(-1))
        assert o.claim_info(cid) == p.claim_info(cid)
    assert not o.offload(ids[4:]).any()                                        # later call dedups against the store
    d2 = set(k for cid in ids for k in keys[cid])
    assert o.stats()["host_used"] == len(d2) * g.blk_bytes == o.link_bytes()[0]
    used, _ = o.pool_state()
    view[:, used == 0, :] = W.POISON
    # restore in two calls; a BITFLIP on a shared block of claim 0 must not touch claim 2 (same group, same block)
    o.set_faults([(ids[0], W.FK_BITFLIP, 5 * g.blk_bytes + 17)])
    st = o.restore(ids[:3])
    assert list(st) == [8, 0, 0]
    expect_h2d = len(keys[ids[0]]) + len(set(keys[ids[1]]) | set(keys[ids[2]]))
    assert o.link_bytes()[1] == expect_h2d * g.blk_bytes
    held = set(k for cid in ids[3:] for k in keys[cid])
    assert o.stats()["host_used"] == len(held) * g.blk_bytes
    assert not o.restore(ids[3:]).any()
    assert o.stats()["host_used"] == 0
    for cid in ids[1:]:
        bt = o.claim_blocks(cid)
        assert np.array_equal(view[:, bt, :].transpose(1, 0, 2), before[cid])   # bit-exact round trip
    ev = o.outcomes()
    ok, why = V.validate(ev)
    assert ok, why
    assert V.failure_outcome_gate(ev, ids[0]) and all(V.observation_gate(ev, c) for c in ids[1:])


def test_dedup_events_and_statuses_equal_the_plain_store():
    a, wl, wave, va, ids = build(True)
    b, _, _, vb, _ = build(False)
    for o, view in ((a, va), (b, vb)):
        o.offload(ids)
        used, _ = o.pool_state()
        view[:, used == 0, :] = W.POISON
        o.set_faults([(ids[2], W.FK_XFER_ERROR, 0)])
        o.restore(ids)
    assert np.array_equal(a.outcomes(), b.outcomes())
    assert np.array_equal(va, vb)
    assert a.link_bytes()[0] < b.link_bytes()[0] and a.link_bytes()[1] < b.link_bytes()[1]
    assert a.set_dedup(False) == 0                                             # allowed again: nothing is held


def test_dedup_host_space_is_granted_by_worst_case_then_charged_by_content():
    o, wl, wave, view, ids = build(True, host=70 * W.GEOMS[0].blk_bytes)
    st = o.offload(ids)
    # SURVEY 8(c).2 offload: claims are served in batch order while the running sum of nb*blk fits the host store
    # that was free at call entry -- every block counted as new; the first claim that does not fit and all later ones
    # get NO_HOST_SPACE
    assert list(st[:2]) == [0, 0] and 7 in list(st)
    first_refused = list(st).index(7)
    assert all(s == 7 for s in st[first_refused:])                              # prefix rule (R7) unchanged
    assert o.stats()["host_used"] <= 70 * wl.geom.blk_bytes
    assert o.set_dedup(False) != 0                                             # refused while bytes are held


def _three_claims(host_blocks, dedup):
    """Tiny geometry; claims 1 and 2 name the SAME 28 physical blocks (identical content), claim 3 names 28 others."""
    g = W.GEOMS[0]
    pool = W.pool_host(g)
    fill = np.zeros(g.pool_blocks, np.uint8)
    fill[:56] = g.block_size
    o = rco.Oracle(g.layers, g.kv_heads, g.head_dim, g.elem_bytes, g.block_size, g.pool_blocks, pool, fill,
                   host_blocks * g.blk_bytes)
    assert o.set_dedup(dedup) == 0
    o.mark_used(np.arange(56))
    t = list(range(28))
    assert not o.accept([1, 2, 3], [448] * 3, [448] * 3, [0, 28, 56, 84], t + t + list(range(28, 56))).any()
    assert not o.materialize([1, 2, 3]).any()
    return o, g


def test_dedup_grant_rule_is_the_call_entry_prefix_sum_not_the_content_charge():
    """The one input on which the two candidate grant rules differ.  Rule taken (DESIGN 11, from
    SURVEY 8(c).2 "served while the running sum of nb*blk fits the free host store ... a pure prefix-sum rule"): the
    sum counts every block as new, so with room for 83 blocks the third claim (28+28+28 = 84) is refused although the
    store would hold only 56 blocks afterwards.  A content-charged grant (host_used as it stands at the claim's turn
    + nb*blk: 28 + 28 = 56 <= 83) would serve it."""
    o, g = _three_claims(83, True)
    assert o.offload([1, 2, 3]).tolist() == [0, 0, 7]
    assert o.stats()["host_used"] == 28 * g.blk_bytes and o.link_bytes()[0] == 28 * g.blk_bytes   # charged by content
    assert o.offload([3]).tolist() == [0]                  # a later call sees what is really held: 28 + 28 <= 83
    assert o.stats()["host_used"] == 56 * g.blk_bytes
    o, g = _three_claims(84, True)
    assert o.offload([1, 2, 3]).tolist() == [0, 0, 0]
    o, g = _three_claims(83, False)                        # the plain store agrees on the statuses: same rule, R7
    assert o.offload([1, 2, 3]).tolist() == [0, 0, 7]
    assert o.stats()["host_used"] == 56 * g.blk_bytes
