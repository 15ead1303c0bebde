"""NEXT-3 pins: multi-claim reuse requests with exact blocking_claim_ids, and the other claim-scoped
outcomes of a failed restoration (demotion, expiry).

P:L384  path C: only the target claim is named; the non-target restores, 0 failure attributions
P:L87   blocking_claim_ids attribute the action to the resident claim(s) that caused it
P:L269  "smear blocking ids across claims" -> ambiguous or smeared attribution fails closed
P:L105/P:L120  offloadable: "claim-scoped restoration failure/refusal, demotion, expiry ... when restoration fails"
P:L267  the failure outcome is emitted before fallback or terminal handling
"""
import itertools

import numpy as np

from conftest import build_tiny_oracle
from oracle import rco, validator as V
from paper_2606_01387_b200 import workloads as W

F = V.REQ_FLAG


def prepared(faults):
    o, wl, wave, pool, fill = build_tiny_oracle()
    ids = [c.claim_id for c in wl.claims]
    o.accept(ids, [c.P for c in wl.claims], [c.N for c in wl.claims], wave.bt_off, wave.bt_ids)
    o.materialize(ids)
    o.offload(ids)
    HIST[0] = o.outcomes()
    assert o.set_faults(faults) == 0
    return o, ids


HIST = [None]


def whole(ev):
    """The stream from the start: acceptance precedes every lifecycle record."""
    return np.concatenate([HIST[0], ev])


def test_request_refusal_names_exactly_the_failed_subset():
    o, ids = prepared([])
    o.set_faults([(ids[1], W.FK_XFER_ERROR, 0), (ids[4], W.FK_BITFLIP, 99)])
    req = 0xABCDEF
    st = o.restore_request(req, ids[:6])
    assert list(st) == [0, 8, 0, 0, 8, 0]
    ev = o.outcomes()
    ok, why = V.validate(whole(ev))
    assert ok, why
    grp = [e for e in ev if int(e["code"]) == 8]
    assert [int(e["claim_id"]) for e in grp] == [ids[1], ids[4]]                    # blocking_claim_ids, batch order
    assert all(int(e["arg"]) == req and int(e["aux"]) == (F | 2) for e in grp)
    assert [int(e["seq"]) for e in grp] == [int(ev["seq"][-2]), int(ev["seq"][-1])]  # one run, after the per-claim records
    for k in (0, 2, 3, 5):                                                          # non-targets restored, 0 attributions
        codes = [int(e["code"]) for e in ev if int(e["claim_id"]) == ids[k]]
        assert codes == [4, 6]
    for k in (1, 4):
        assert [int(e["code"]) for e in ev if int(e["claim_id"]) == ids[k]] == [4, 5, 7, 8]
        assert o.claim_info(ids[k])["state"] == 5
    assert o.restore_request(req, ids[:6]).tolist() == [3] * 6                      # nothing left to restore: BAD_STATE


def test_request_without_failure_emits_no_refusal_and_single_failure_is_a_group_of_one():
    o, ids = prepared([])
    st = o.restore_request(7, ids[:3])
    ev = o.outcomes()
    assert not st.any() and 8 not in [int(e["code"]) for e in ev] and V.validate(whole(ev))[0]
    HIST[0] = whole(ev)
    o.set_faults([(ids[4], W.FK_XFER_ERROR, 0)])
    o.restore_request(8, ids[3:6])
    ev = o.outcomes()
    g = [e for e in ev if int(e["code"]) == 8]
    assert len(g) == 1 and int(g[0]["claim_id"]) == ids[4] and int(g[0]["aux"]) == (F | 1) and int(g[0]["arg"]) == 8
    assert V.validate(whole(ev))[0]


def test_smeared_or_incomplete_blocking_ids_fail_closed():
    o, ids = prepared([])
    o.set_faults([(ids[1], W.FK_XFER_ERROR, 0), (ids[4], W.FK_XFER_ERROR, 0)])
    o.restore_request(5, ids[:6])
    full = o.outcomes()
    ev = whole(full)
    assert V.validate(ev)[0]
    n = ev.size
    smear = ev.copy(); smear["claim_id"][n - 1] = ids[0]            # names a claim that restored fine
    assert not V.validate(smear)[0]
    short = ev.copy(); short["aux"][n - 2:] = F | 1                  # claims a subset of one while two failed
    assert not V.validate(short)[0]
    dropped = np.delete(ev, n - 1)                                   # a prefix is still a prefix ...
    assert V.validate(dropped)[0]
    extra = np.zeros(1, ev.dtype); extra["seq"], extra["claim_id"], extra["code"] = n + 5, ids[0], V.USE
    assert not V.validate(np.concatenate([dropped, extra]))[0]       # ... but nothing may interrupt the run
    other = ev.copy(); other["arg"][n - 1] = 6                       # second record under another request id
    assert not V.validate(other)[0]
    classic = ev.copy(); classic["aux"][n - 2:] = 1                  # per-claim form must carry [C] itself
    assert not V.validate(classic)[0]


def test_all_interleavings_of_a_two_failure_request():
    """Brute force: claims A and B each RESTORE_REQUIRED, LOAD_FAILED, RESTORATION_FAILED, REFUSED(group of 2).
    An order-preserving interleaving is accepted iff both RESTORATION_FAILED precede the run and the run is contiguous."""
    A, B, req = 11, 22, 9
    pre = [(0, c, code, 0, 0) for c in (A, B) for code in (1, 2, 3)]
    seq = {A: [(4, 0, 0), (5, 0, 0), (7, 0, 0), (8, F | 2, req)], B: [(4, 0, 0), (5, 0, 0), (7, 0, 0), (8, F | 2, req)]}
    n_ok = 0
    for pos in itertools.combinations(range(8), 4):
        order = [A if i in pos else B for i in range(8)]
        it = {A: iter(seq[A]), B: iter(seq[B])}
        tail = [(0, c) + next(it[c]) for c in order]
        ev = [(i, c, code, aux, arg) for i, (_, c, code, aux, arg) in enumerate(pre + tail)]
        codes = [(c, code) for _, c, code, _, _ in ev[6:]]
        refs = [i for i, x in enumerate(codes) if x[1] == 8]
        rfs = [i for i, x in enumerate(codes) if x[1] == 7]
        want = max(rfs) < min(refs) and refs[1] == refs[0] + 1
        assert V.validate(ev)[0] == want, order
        n_ok += want
    assert n_ok == 2 * 20           # the two RF-prefixes interleave freely (C(6,3) = 20), the run comes last in either order


def test_demotion_and_expiry_are_ordered_claim_scoped_outcomes():
    o, ids = prepared([])
    assert o.set_policy([ids[0], ids[1]], [1, 2]) == 0
    assert o.set_policy([12345], [1]) != 0 and o.set_policy([ids[2]], [3]) != 0
    o.set_faults([(ids[0], W.FK_XFER_ERROR, 0), (ids[1], W.FK_BITFLIP, 3), (ids[2], W.FK_XFER_ERROR, 0)])
    st = o.restore_request(77, ids[:4])
    assert list(st) == [8, 8, 8, 0]
    ev = o.outcomes()
    assert V.validate(whole(ev))[0]
    by = {c: [int(e["code"]) for e in ev if int(e["claim_id"]) == c] for c in ids[:4]}
    assert by[ids[0]] == [4, 5, 7, 9] and by[ids[1]] == [4, 5, 7, 10]               # demoted / expired right after the failure
    assert by[ids[2]] == [4, 5, 7, 8] and by[ids[3]] == [4, 6]
    g = [e for e in ev if int(e["code"]) == 8]
    assert len(g) == 1 and int(g[0]["aux"]) == (F | 1) and int(g[0]["claim_id"]) == ids[2]   # only the refusing claim blocks
    assert [o.claim_info(c)["state"] for c in ids[:3]] == [6, 7, 5]
    assert list(o.offload(ids[:3])) == [3, 3, 3] and list(o.restore(ids[:3])) == [3, 3, 3]   # terminal
    fin = np.zeros(1, ev.dtype); fin["seq"], fin["claim_id"], fin["code"] = 10 ** 6, ids[0], V.REQUEST_FINISHED
    hist = HIST[0]
    allv = np.concatenate([hist, ev, fin]); allv["seq"] = np.arange(allv.size)
    assert V.validate(allv)[0]                                                       # terminal handling after the outcome
    early = np.concatenate([hist, ev[: list(ev["code"]).index(9)], fin, ev[list(ev["code"]).index(9):]])
    early["seq"] = np.arange(early.size)
    assert not V.validate(early)[0]                                                  # ... never before it


def test_plain_restore_is_unchanged_by_the_extension():
    o, ids = prepared([])
    o.set_faults([(ids[3], W.FK_XFER_ERROR, 0)])
    o.restore(ids)
    ev = o.outcomes()
    g = [e for e in ev if int(e["code"]) == 8]
    assert len(g) == 1 and int(g[0]["aux"]) == 1 and int(g[0]["arg"]) == ids[3] == int(g[0]["claim_id"])
