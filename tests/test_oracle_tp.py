"""NEXT-4 pins: the TP-sharded restore of the oracle (DESIGN.md 8 / R24).  The pool is split by kv_head
over 2 ranks; each rank is an oracle over its shard.  Pinned: the merged verdict is the AND of the ranks' verdicts with
bad = min over the failing ranks; every rank emits the byte-identical stream; it equals the unsharded oracle's stream
in (seq, claim, code, aux); a claim that verified locally but failed elsewhere is refused and its blocks freed on every
rank (P:L384 attribution survives, P:L269 no smearing); the restored shards reassemble to the unsharded pool."""
import numpy as np
import pytest

from oracle import rco, validator as V
from paper_2606_01387_b200 import tp

import tp_inputs as T

XFER, FLIP = 1, 2


def oracles():
    full, tabs, fill = T.make()
    parts = [T.shard(full, r).copy() for r in range(T.G)]
    fills = [np.zeros(T.NB, np.uint8) for _ in range(T.G)]
    os_ = [rco.Oracle(T.L, T.H // T.G, T.D, T.E, T.BS, T.NB, parts[r], fills[r]) for r in range(T.G)]
    for o in os_:
        assert o.set_tp(T.G) == 0
    ffull = np.zeros(T.NB, np.uint8)
    whole = rco.Oracle(T.L, T.H, T.D, T.E, T.BS, T.NB, full, ffull)
    ids = None
    for o, f in zip(os_ + [whole], fills + [ffull]):
        ids = T.admit(o, tabs, f, fill)
    return os_, parts, whole, full, ids


def tp_round(os_, ids, faults):
    """faults[r] = fault list of rank r.  Returns the per-rank statuses."""
    loc, sts = [], []
    for o, f in zip(os_, faults):
        assert o.set_faults(f) == 0
        st, v = o.tp_restore_verify(ids)
        sts.append(st)
        loc.append(v)
    gathered = np.stack(loc)
    return [o.tp_restore_commit(gathered, st) for o, st in zip(os_, sts)], gathered


def test_tp_sharded_restore_common_verdict_and_identical_streams():
    os_, parts, whole, full, ids = oracles()
    before = full.copy()
    for o in os_ + [whole]:
        assert not o.offload(ids).any()
    blk = os_[0].blk
    # claim 0: clean.  claim 1: transfer error on rank 1 only.  claim 2: bit flip in block 5 on rank 0 and block 2 on
    # rank 1 -> bad = 2.  claim 3: transfer error on rank 0, bit flip in block 4 on rank 1 -> bad = 4.  claim 4: clean.
    f0 = [(ids[2], FLIP, 5 * blk + 17), (ids[3], XFER, 0)]
    f1 = [(ids[1], XFER, 0), (ids[2], FLIP, 2 * blk + 99), (ids[3], FLIP, 4 * blk)]
    sts, gathered = tp_round(os_, ids, [f0, f1])
    assert [list(s) for s in sts] == [[0, 8, 8, 8, 0]] * 2                       # the SAME statuses on every rank
    assert gathered["flags"].tolist() == [[3, 3, 1, 1, 3], [3, 1, 1, 1, 3]]      # rank 0 verified claim 1 locally
    ev = [o.outcomes() for o in os_]
    assert ev[0].tobytes() == ev[1].tobytes()                                    # byte-identical streams
    ok, why = V.validate(ev[0])
    assert ok, why
    lf = {int(e["claim_id"]): int(e["aux"]) for e in ev[0] if int(e["code"]) == 5}
    assert lf == {ids[1]: 0xFFFFFFFF, ids[2]: 2, ids[3]: 4}
    assert all(int(e["arg"]) == 0 for e in ev[0] if int(e["code"]) in (3, 6))    # no rank-local chain in the stream
    for o in os_:                                                                # refused everywhere, blocks freed everywhere
        assert [o.claim_info(c)["state"] for c in ids] == [4, 5, 5, 5, 4]
        used, ref = o.pool_state()
        assert int(used.sum()) == int(ref.sum()) == sum(o.claim_info(c)["nb"] for c in (ids[0], ids[4]))
    assert np.array_equal(os_[0].pool_state()[0], os_[1].pool_state()[0])
    assert all(np.array_equal(os_[0].claim_blocks(c), os_[1].claim_blocks(c)) for c in ids)
    # the unsharded oracle with the union of the faults: same records up to the rank-local chain
    whole.set_faults([(ids[1], XFER, 0), (ids[2], FLIP, 2 * whole.blk + 5), (ids[3], FLIP, 4 * whole.blk)])
    assert list(whole.restore(ids)) == [0, 8, 8, 8, 0]
    ew = whole.outcomes()
    for f in ("seq", "claim_id", "code", "aux"):
        assert np.array_equal(ew[f], ev[0][f]), f
    # restored shards reassemble to the unsharded pool, block for block, in the same (lowest free) block ids
    re = T.unshard(parts).reshape(T.L * 2, T.NB, -1)
    wv = full.reshape(T.L * 2, T.NB, -1)
    for c in (ids[0], ids[4]):
        bt = whole.claim_blocks(c)
        assert np.array_equal(re[:, bt, :], wv[:, bt, :])


def test_tp_merge_rules_and_disagreement():
    os_, parts, whole, full, ids = oracles()
    for o in os_:
        assert not o.offload(ids[:3]).any()
    sts, loc = [], []
    for o in os_:
        st, v = o.tp_restore_verify(ids[:3])
        assert list(st) == [-1, -1, -1] and v["flags"].tolist() == [3, 3, 3]       # served: decided by the commit
        with pytest.raises(ValueError):
            o.tp_restore_verify(ids[:3])                                         # one split restore at a time
        sts.append(st)
        loc.append(v)
    bad = np.stack(loc)
    bad["flags"][1][2] = 0                                                       # rank 1 claims it did not serve claim 2
    with pytest.raises(ValueError):
        os_[0].tp_restore_commit(bad, sts[0])
    with pytest.raises(ValueError):
        os_[0].tp_restore_commit(np.stack(loc)[:, :2], sts[0])                   # wrong batch size
    n0 = os_[0].stats()["n_events"]
    assert n0 == 5 + 5 + 3                                                        # nothing emitted by verify or by the rejects
    g = np.stack(loc)
    g["flags"][1][1] = 1                                                         # rank 1 failed claim 1 in block 7
    g["bad"][1][1] = 7
    for o, st in zip(os_, sts):
        assert list(o.tp_restore_commit(g, st)) == [0, 8, 0]
    ev = os_[0].outcomes()
    assert [int(e["aux"]) for e in ev if int(e["code"]) == 5] == [7]
    assert os_[0].outcomes().size == 0 and ev.tobytes() == os_[1].outcomes().tobytes()
    # G = 1 degenerates to the plain restore
    one = rco.Oracle(T.L, T.H, T.D, T.E, T.BS, T.NB, full.copy(), np.zeros(T.NB, np.uint8))
    _, tabs, fill = T.make()
    T.admit(one, tabs, one.fill, fill)
    assert not one.offload(ids).any()
    one.set_faults([(ids[3], XFER, 0)])
    st, v = one.tp_restore_verify(ids)
    assert list(one.tp_restore_commit(tp.all_gather_verdicts(v), st)) == [0, 0, 0, 8, 0]
    whole.offload(ids); whole.set_faults([(ids[3], XFER, 0)]); whole.restore(ids)
    assert one.outcomes().tobytes() == whole.outcomes().tobytes()


def test_merge_outcomes_of_claim_sharded_replicas_keeps_attribution():
    """streams of independent replicas joined by (gpu, seq): the merged stream validates, every claim
    keeps its own order, and the gates name the same claims as before the merge."""
    import trace_inputs as TI
    a, b = TI.make_trace(300, 11), TI.make_trace(300, 12)
    b = b[~np.isin(b["claim_id"], a["claim_id"])]
    merged, origin = tp.merge_outcomes([a, b])
    assert V.validate(merged)[0] and merged.size == a.size + b.size
    assert origin["gpu"].tolist() == [0] * a.size + [1] * b.size and np.array_equal(origin["seq"][:a.size], a["seq"])
    for src in (a, b):
        for cid in np.unique(src["claim_id"])[:40]:
            assert V.failure_outcome_gate(merged, int(cid)) == V.failure_outcome_gate(src, int(cid))
            assert V.observation_gate(merged, int(cid)) == V.observation_gate(src, int(cid))
    bad = a.copy()
    bad["seq"][5] = bad["seq"][4]
    with pytest.raises(AssertionError):
        tp.merge_outcomes([bad])


def test_numa_helpers_parse_and_never_fail_without_a_gpu():
    assert tp.parse_cpulist("0-3,8,10-11\n") == {0, 1, 2, 3, 8, 10, 11}
    assert tp.bind_to_gpu_numa_node(0) in (None, 0, 1, 2, 3)
