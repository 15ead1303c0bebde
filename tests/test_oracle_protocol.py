"""Pins for the oracle's protocol part against what the paper prints.

P:L27   the seven-step accepted order of the running example (failure path)
P:L360-367 path A (success), incl. hit=448
P:L371-380 path B
P:L384  path C: target-only attribution
P:L25: wrong-claim / unclaimed failure, ordinary offload,
        fallback recompute, restore-after-use are not accepted
P:L337  injection semantics;  P:L199 ambiguity fails closed (no event on error)
"""
import numpy as np
import pytest

from conftest import build_tiny_oracle
from oracle import rco, validator as V
from paper_2606_01387_b200 import workloads as W

GOLD = [l.split("#")[0].strip() for l in open(__file__.rsplit("/", 1)[0] + "/golden/event_orders.txt")]
GOLD = {l.split(":")[0].strip(): [x.strip() for x in l.split(":")[1].split(",")] for l in GOLD if l}
CODE = {v: k for k, v in rco.EV_NAMES.items()}


def names(ev, cid):
    return [rco.EV_NAMES[int(e["code"])] for e in ev if int(e["claim_id"]) == cid]


def run_tiny(fault_kind=W.FK_BITFLIP):
    o, wl, wave, pool, fill = build_tiny_oracle()
    ids = [c.claim_id for c in wl.claims]
    before = {c.claim_id: None for c in wl.claims}
    st_a = o.accept(ids, [c.P for c in wl.claims], [c.N for c in wl.claims], wave.bt_off, wave.bt_ids)
    st_m = o.materialize(ids)
    logical = {}
    g = wl.geom
    view = pool.reshape(2 * g.layers, g.pool_blocks, g.page_bytes)
    for c in wl.claims:
        bt = o.claim_blocks(c.claim_id)
        logical[c.claim_id] = view[:, bt, :].transpose(1, 0, 2).copy()     # [block][page g][bytes]
    st_o = o.offload(ids)
    host = {c.claim_id: o.host_read(c.claim_id) for c in wl.claims}
    used, _ = o.pool_state()
    view[:, used == 0, :] = W.POISON
    faults = [(cid, fault_kind, p) for cid, _, p in wave.faults]
    assert o.set_faults(faults) == 0
    st_r = o.restore(ids)
    return o, wl, wave, pool, (st_a, st_m, st_o, st_r), logical, host


@pytest.mark.parametrize("kind", [W.FK_BITFLIP, W.FK_XFER_ERROR])
def test_tiny_streams_match_the_papers_orders(kind):
    o, wl, wave, pool, (st_a, st_m, st_o, st_r), logical, host = run_tiny(kind)
    ev = o.outcomes()
    ok, why = V.validate(ev)
    assert ok, why
    assert list(ev["seq"]) == list(range(len(ev)))
    for k, c in enumerate(wl.claims):
        got = names(ev, c.claim_id)
        if k == 6:      # 400 tokens < 448: predicate false -> accepted only, no lifecycle events
            assert got == ["ACCEPTED"] and st_m[k] == 1 and st_o[k] == 3 and st_r[k] == 3
        elif k == 3:    # P:L27 seven steps, exact
            assert got == GOLD["failure_path"] and st_r[k] == 8
            assert V.failure_outcome_gate(ev, c.claim_id) and not V.observation_gate(ev, c.claim_id)
            ref = [e for e in ev if int(e["claim_id"]) == c.claim_id and int(e["code"]) == 8][0]
            assert int(ref["arg"]) == c.claim_id and int(ref["aux"]) == 1       # blocking_claim_ids=[C]
            lf = [e for e in ev if int(e["claim_id"]) == c.claim_id and int(e["code"]) == 5][0]
            if kind == W.FK_XFER_ERROR:
                assert int(lf["aux"]) == 0xFFFFFFFF
            else:
                nbytes = o.claim_info(c.claim_id)["nb"] * wl.geom.blk_bytes
                assert int(lf["aux"]) == (c.fault[1] % nbytes) // wl.geom.blk_bytes   # affected block evidence
        else:           # path A
            assert got == GOLD["success_path"] and st_r[k] == 0
            assert V.observation_gate(ev, c.claim_id) and not V.failure_outcome_gate(ev, c.claim_id)
            rr = [e for e in ev if int(e["claim_id"]) == c.claim_id and int(e["code"]) == 4][0]
            assert int(rr["aux"]) == c.M                                          # lookup hit = M
    # claim-major batch order inside one call: each claim's restore events are consecutive
    rest = [int(e["claim_id"]) for e in ev if int(e["code"]) >= 4]
    runs = [rest[0]] + [b for a, b in zip(rest, rest[1:]) if a != b]
    assert len(runs) == len(set(runs))


def test_hit_448_is_served():
    # hit=448 against leading-prefix-at-least-448 is served (">=")
    wl = W.make_workload(0)
    wl.claims = wl.claims[:1]
    wl.claims[0].P, wl.claims[0].M, wl.claims[0].fault = 460, 448, None
    o, wl, wave, pool, fill = build_tiny_oracle(wl)
    c = wl.claims[0]
    assert o.accept([c.claim_id], [c.P], [c.N], wave.bt_off, wave.bt_ids)[0] == 0
    assert o.materialize([c.claim_id])[0] == 0
    assert o.offload([c.claim_id])[0] == 0 and o.restore([c.claim_id])[0] == 0
    ev = o.outcomes()
    assert [int(e["aux"]) for e in ev if int(e["code"]) in (2, 4)] == [448, 448]
    assert o.claim_info(c.claim_id)["nb"] == 28                                  # 28 blocks of 16


def test_round_trip_is_bit_exact_and_host_copy_survives_bitflip():
    o, wl, wave, pool, st, logical, host = run_tiny(W.FK_BITFLIP)
    g = wl.geom
    view = pool.reshape(2 * g.layers, g.pool_blocks, g.page_bytes)
    for k, c in enumerate(wl.claims):
        if k in (3, 6):
            continue
        info = o.claim_info(c.claim_id)
        bt = o.claim_blocks(c.claim_id)
        assert len(bt) == info["nb"]
        now = view[:, bt, :].transpose(1, 0, 2)
        assert np.array_equal(now, logical[c.claim_id][: info["nb"]])
        # offload bytes = independent fancy-index gather, block-major then page
        assert np.array_equal(host[c.claim_id], logical[c.claim_id][: info["nb"]].reshape(-1))
    # the bit-flipped claim's host copy was intact when read before restore
    c3 = wl.claims[3]
    nb3 = (c3.M + g.block_size - 1) // g.block_size
    assert np.array_equal(host[c3.claim_id], logical[c3.claim_id][:nb3].reshape(-1))
    used, ref = o.pool_state()
    live = sum(len(o.claim_blocks(c.claim_id)) for c in wl.claims if o.claim_info(c.claim_id)["state"] == 4)
    assert int(ref.sum()) == live + int(ref[o.claim_blocks(wl.claims[6].claim_id)].sum())


def test_target_only_attribution_path_c():
    # two claims, one process; only the target is named, the other restores
    wl = W.make_workload(0)
    wl.claims = wl.claims[:2]
    for c in wl.claims:
        c.fault = None
    o, wl, wave, pool, fill = build_tiny_oracle(wl)
    a, b = wl.claims[0].claim_id, wl.claims[1].claim_id
    ids = [a, b]
    o.accept(ids, [c.P for c in wl.claims], [c.N for c in wl.claims], wave.bt_off, wave.bt_ids)
    o.materialize(ids); o.offload(ids)
    o.set_faults([(b, W.FK_XFER_ERROR, 0)])
    assert list(o.restore(ids)) == [0, 8]
    ev = o.outcomes()
    assert V.observation_gate(ev, a) and V.failure_outcome_gate(ev, b)
    assert all(int(e["claim_id"]) == b for e in ev if int(e["code"]) in (5, 7, 8))


def test_wrong_claim_unclaimed_and_disabled_injection_change_nothing():
    wl = W.make_workload(0)
    wl.claims = wl.claims[:2]
    for c in wl.claims:
        c.fault = None
    o, wl, wave, pool, fill = build_tiny_oracle(wl)
    a, b = wl.claims[0].claim_id, wl.claims[1].claim_id
    o.accept([a, b], [c.P for c in wl.claims], [c.N for c in wl.claims], wave.bt_off, wave.bt_ids)
    o.materialize([a, b]); o.offload([a, b])
    assert o.set_faults([(0, W.FK_XFER_ERROR, 0)]) != 0                  # unclaimed needs the separate flag
    assert o.set_faults([(0xABCDEF, W.FK_XFER_ERROR, 0), (b, W.FK_BITFLIP, 3), (0, W.FK_XFER_ERROR, 0)], 1) == 0
    assert list(o.restore([a])) == [0]                                   # wrong-claim + unclaimed: a unaffected
    ev = o.outcomes()
    assert V.observation_gate(ev, a) and names(ev, b)[-1] == "OFFLOADED"
    assert o.stats()["generic_failures"] == 1                            # counter only, no event
    assert o.set_faults([]) == 0                                         # disarm: injection off by default
    assert list(o.restore([b])) == [0]


def test_illegal_calls_emit_nothing():
    o, wl, wave, pool, fill = build_tiny_oracle()
    c = wl.claims[0]
    n0 = o.stats()["n_events"]
    for fn in (o.materialize, o.offload, o.restore, o.release):
        assert list(fn([c.claim_id])) == [2]                             # post-hoc naming: unknown claim
    bt = wave.bt_ids[wave.bt_off[0]:wave.bt_off[1]]
    off = [0, len(bt)]
    assert o.accept([0], [c.P], [c.N], off, bt)[0] == 2                  # id 0 reserved
    assert o.accept([7], [c.P], [c.P + 1], off, bt)[0] == 5              # N > P
    assert o.accept([7], [c.P], [0], off, bt)[0] == 5
    assert o.accept([7], [c.P + 16], [c.N], off, bt)[0] == 5             # table length != ceil(P/BS)
    bad = bt.copy(); bad[1] = bad[0]
    assert o.accept([7], [c.P], [c.N], off, bad)[0] == 5                 # repeated id
    bad = bt.copy(); bad[0] = 256
    assert o.accept([7], [c.P], [c.N], off, bad)[0] == 5                 # out of range
    o.mark_free([int(bt[2])])
    assert o.accept([7], [c.P], [c.N], off, bt)[0] == 5                  # block not in use
    o.mark_used([int(bt[2])])
    assert o.stats()["n_events"] == n0
    assert o.accept([7, 7], [c.P, c.P], [c.N, c.N], [0, len(bt), 2 * len(bt)], np.concatenate([bt, bt])).tolist() == [0, 4]
    assert o.offload([7])[0] == 3 and o.restore([7])[0] == 3             # ordinary offload w/o materialized claim
    assert o.materialize([7])[0] == 0 and o.materialize([7])[0] == 3
    assert o.restore([7])[0] == 3                                        # restore before offload
    assert o.offload([7, 7]).tolist() == [0, 3]
    assert o.restore([7, 7]).tolist() == [0, 3]                          # double restore (restore-after-use)
    assert o.restore([7])[0] == 3
    assert names(o.outcomes(), 7) == GOLD["success_path"]
    # after refusal the claim is terminal: no fallback "restored"
    assert o.offload([7])[0] == 0
    o.set_faults([(7, W.FK_XFER_ERROR, 0)])
    assert o.restore([7])[0] == 8
    for fn in (o.materialize, o.offload, o.restore):
        assert fn([7])[0] == 3
    assert V.failure_outcome_gate(o.outcomes(), 7) is False              # 7's stream was drained in two parts
