"""NEXT-3 GPU parity: rc_protect / rc_make_room / rc_protected_map (k_vic_posmax, k_vic_gain, k_vic_decide, k_prot_map,
k_emit in its DEMOTE / CONFLICT modes) against the oracle: status, ids, events, allocator state, claim states and the
protected footprint after every call (DESIGN.md 12 / R23)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import validator as V
from paper_2606_01387_b200 import rc, workloads as W
from parity_harness import Pair
from shared_tiny import make_shared_tiny


def admit(p, wl, wave):
    o, r = p.o, p.r
    ids = [c.claim_id for c in wl.claims]
    p.set_fill(wave.fill_ids, wave.fill_val)
    for x in (o, r):
        assert x.mark_used(wave.used_ids) == 0
    args = (ids, [c.P for c in wl.claims], [c.N for c in wl.claims], wave.bt_off, wave.bt_ids)
    assert np.array_equal(o.accept(*args), r.accept(*args))
    assert np.array_equal(o.materialize(ids), r.materialize(ids))
    return ids


def both(p, fn, *a):
    ra, rb = getattr(p.o, fn)(*a), getattr(p.r, fn)(*a)
    assert ra == rb, (fn, a, ra, rb)
    return ra


def check(p, ids, what):
    p.check_claims(ids, what, digests=False)
    p.check_pool_state(what, bytes_too=False)
    assert np.array_equal(p.o.protected_map(), p.r.protected_map()), what


def test_make_room_tiny_every_branch():
    wl = W.make_workload(0)
    for c in wl.claims:
        c.M, c.fault = c.P, None
    p = Pair(wl, 1 << 30, chunk_blocks=16)
    wave = W.plan_waves(wl, 1 << 30)[0]
    ids = admit(p, wl, wave)
    free = 256 - wave.used_ids.size
    assert both(p, "make_room", 9, free) == (0, [])                       # fits
    assert both(p, "protect", [ids[1], ids[4]], [1, 1]) == 0
    assert both(p, "protect", [0xBAD], [1]) != 0
    check(p, ids, "protect")
    st, got = both(p, "make_room", 10, free + 40)                         # demotes claims 0 and 2 (1 is protected)
    assert st == 0 and got == [ids[0], ids[2]]
    check(p, ids, "evict")
    assert np.array_equal(p.o.offload(ids[:3]), p.r.offload(ids[:3]))     # demoted claims are terminal: BAD_STATE
    check(p, ids, "offload after eviction")
    st, got = both(p, "make_room", 11, 256)                               # the whole pool: only protected footprints remain
    assert st == rc.ST_PROTECTED_CONFLICT and got == [ids[4]]             # claim 1 was offloaded: it holds no table
    check(p, ids, "conflict")
    assert both(p, "protect", [ids[4]], [0]) == 0
    st, got = both(p, "make_room", 12, 256)
    assert st == 0 and ids[4] in got
    check(p, ids, "after unprotect")
    p.poison_free()
    assert np.array_equal(p.o.restore([ids[1]]), p.r.restore([ids[1]]))   # protection follows the claim through restore
    check(p, ids, "restore protected")
    assert p.r.protected_map().sum() == p.r.claim_info(ids[1])["nb"]
    st, got = both(p, "make_room", 13, 256)
    assert st == rc.ST_PROTECTED_CONFLICT and got == [ids[1]]
    ev = p.check_events("make_room")
    ok, why = V.validate(ev)
    assert ok, why
    assert [int(e["code"]) for e in ev if int(e["code"]) in (9, 11)].count(11) == 2
    rcode = p.r.L.rc_make_room(p.r.h, 0, 1, None, None, 0, None)
    assert rcode == rc.ERR_INVALID
    p.close()


def test_make_room_shared_blocks_and_random_pressure():
    """Shared prefixes (a block is freed by its LAST holder in victim order) and a random walk of protect / make_room /
    offload / restore over 200 claims: every call compared."""
    wl, wave, copies = make_shared_tiny(n_claims=6)
    p = Pair(wl, 1 << 30, chunk_blocks=16)
    ids = admit(p, wl, wave)
    assert both(p, "protect", [ids[2]], [1]) == 0
    used, _ = p.o.pool_state()
    free = int((used == 0).sum())
    for need in (free + 3, free + 20, free + 60, 256):
        both(p, "make_room", 100 + need, need)
        check(p, ids, "shared need %d" % need)
    ev = p.check_events("shared")
    assert V.validate(ev)[0]
    p.close()

    wl = W.make_workload(0, n_claims=200, pool_blocks=8192)
    for c in wl.claims:
        c.M, c.fault = c.P, None
    p = Pair(wl, 1 << 32, chunk_blocks=256)
    wave = W.plan_waves(wl, 1 << 40)[0]
    ids = admit(p, wl, wave)
    rng = np.random.default_rng(31)
    n_conf = n_evict = 0
    for step in range(40):
        u = rng.random()
        sel = [ids[k] for k in rng.choice(len(ids), 12, replace=False)]
        live = [c for c in sel if p.o.claim_info(c)["state"] in (1, 2, 3, 4)]
        if u < 0.3 and live:
            both(p, "protect", live, [int(x) for x in rng.integers(0, 2, len(live))])
        elif u < 0.45:
            assert np.array_equal(p.o.offload(sel), p.r.offload(sel))
        elif u < 0.6:
            p.poison_free()
            assert np.array_equal(p.o.restore(sel), p.r.restore(sel))
        else:
            used, _ = p.o.pool_state()
            need = int((used == 0).sum()) + int(rng.integers(1, 1500))
            st, got = both(p, "make_room", 7000 + step, need)
            n_conf += st == rc.ST_PROTECTED_CONFLICT
            n_evict += st == 0 and len(got) > 0
        check(p, ids, "random step %d" % step)
    assert n_conf >= 3 and n_evict >= 3
    ev = p.check_events("random pressure")
    ok, why = V.validate(ev)
    assert ok, why
    rep, _ = rc.validate_trace(ev, want_claims=False)
    assert rep["ok"] == 1
    p.close()
