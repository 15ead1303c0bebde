"""NEXT-3 pins: allocator-side protection in the oracle (reading R23).

P:L85  victim_exclusion_before_violation, explicit_conflict_action, blocking_claim_ids, claim_demoted_before_loss
P:L103 hard_protected: "footprint accounting, victim exclusion before violation, an explicit conflict action, blocking
       claim ids ... and order";  P:L270 allocator_hook: "exposes the victim candidate set, protected resident footprint,
       and ordered exclusion or release before predicate-breaking loss"
Pinned here: hand cases for every branch of make_room; the ordered demotion precedes the loss; a refusal names exactly
the protected claims the walk had to enter and evicts nothing; and, by brute force over call sequences on an 8-block
pool, no sequence of calls ever hands a block of a protected footprint to anyone else or changes its bytes.
"""
import numpy as np
import pytest

from oracle import rco, validator as V
from test_oracle_pins import BS4, L_, PAGE, small_oracle

OK, NO_FREE, CONFLICT = 0, 6, 9


def setup(nbp, tables, protect=()):
    """claims 1..n with the given block tables (each block full), accepted in that order and materialized."""
    o, pool, fill = small_oracle(nbp, seed=5)
    blocks = sorted({b for t in tables for b in t})
    o.mark_used(blocks)
    fill[blocks] = BS4
    ids = list(range(1, len(tables) + 1))
    off = np.cumsum([0] + [len(t) for t in tables])
    assert not o.accept(ids, [BS4 * len(t) for t in tables], [1] * len(ids), off, [b for t in tables for b in t]).any()
    assert not o.materialize(ids).any()
    if protect:
        assert o.protect(list(protect), [1] * len(protect)) == 0
    o.ev0 = list(o.outcomes())                           # ACCEPTED / MATERIALIZED records, for whole-stream validation
    return o, pool, fill, ids


def test_make_room_branches():
    # 12 blocks: claims 1..4 hold 2 blocks each (0-7), 4 blocks free
    tabs = [[0, 1], [2, 3], [4, 5], [6, 7]]
    o, *_ = setup(12, tabs)
    assert o.make_room(77, 4) == (OK, []) and len(o.outcomes()) == 0            # fits: nothing happens
    st, ids = o.make_room(77, 7)                                                # 4 free + claims 1, 2 (acceptance order)
    assert (st, ids) == (OK, [1, 2])
    ev = o.outcomes()
    assert [(int(e["claim_id"]), int(e["code"]), int(e["aux"]), int(e["arg"])) for e in ev] == [(1, 9, 2, 77), (2, 9, 2, 77)]
    used, ref = o.pool_state()
    assert used.tolist() == [0, 0, 0, 0, 1, 1, 1, 1, 0, 0, 0, 0] and int(ref.sum()) == 4
    assert o.claim_info(1)["state"] == 6 and o.claim_info(3)["state"] == 2      # demoted is terminal; 3 untouched
    assert o.offload([1])[0] == 3 and o.materialize([1])[0] == 3
    # protected claims are walked last and never evicted
    o, *_ = setup(12, tabs, protect=[1, 3])
    assert o.protected_map().tolist() == [1, 1, 0, 0, 1, 1, 0, 0, 0, 0, 0, 0]
    assert o.make_room(5, 8) == (OK, [2, 4])                                    # the unprotected ones suffice
    ev_all = o.ev0 + list(o.outcomes())
    st, ids = o.make_room(6, 9)                                                 # now only protected footprints are left
    assert (st, ids) == (CONFLICT, [1])                                         # the walk had to enter claim 1 only
    ev = o.outcomes()
    assert [(int(e["claim_id"]), int(e["code"]), int(e["aux"]), int(e["arg"])) for e in ev] == [(1, 11, V.REQ_FLAG | 1, 6)]
    st, ids = o.make_room(7, 12)
    assert (st, ids) == (CONFLICT, [1, 3])
    st, ids = o.make_room(8, 13)                                                # more than the pool: all protected named
    assert (st, ids) == (CONFLICT, [1, 3])
    used, ref = o.pool_state()
    assert used[:2].all() and used[4:6].all() and int(ref.sum()) == 4           # nothing was evicted by the refusals
    assert o.claim_info(1)["state"] == 2 and o.claim_info(3)["state"] == 2
    ok, why = V.validate(ev_all + list(ev) + list(o.outcomes()))
    assert ok, why
    # all-or-nothing: when the unprotected victims do not suffice, they are NOT evicted either
    o, *_ = setup(12, tabs, protect=[4])
    st, ids = o.make_room(9, 11)                                                # 4 free + 6 unprotected = 10 < 11
    assert (st, ids) == (CONFLICT, [4])
    assert all(o.claim_info(c)["state"] == 2 for c in (1, 2, 3, 4)) and int(o.pool_state()[1].sum()) == 8
    # no protected footprint in the way: plain exhaustion, no event
    o, *_ = setup(12, tabs)
    assert o.make_room(9, 13) == (NO_FREE, []) and len(o.outcomes()) == 0
    with pytest.raises(ValueError):
        o.make_room(0, 1)                                                       # request id 0 is reserved
    assert o.protect([99], [1]) != 0 and o.protect([1], [2]) != 0


def test_shared_blocks_are_freed_by_their_last_holder_only():
    # claims 1 and 2 share block 0; evicting claim 1 alone frees only block 1
    o, *_ = setup(6, [[0, 1], [0, 2], [3]])
    assert int((o.pool_state()[0] == 0).sum()) == 2                             # blocks 4, 5 free
    assert o.make_room(3, 3) == (OK, [1])                                       # +1 (block 1)
    assert o.pool_state()[0].tolist() == [1, 0, 1, 1, 0, 0]
    o, *_ = setup(6, [[0, 1], [0, 2], [3]])
    assert o.make_room(3, 5) == (OK, [1, 2])                                    # +1, then +2 (blocks 0 and 2)
    assert o.pool_state()[0].tolist() == [0, 0, 0, 1, 0, 0]
    # a block shared with a protected claim is not freed by evicting the unprotected holder
    o, *_ = setup(6, [[0, 1], [0, 2], [3]], protect=[2])
    st, ids = o.make_room(3, 5)                                                 # 2 free + 1 (claim 1) + 1 (claim 3) = 4 < 5
    assert (st, ids) == (CONFLICT, [2])
    assert o.make_room(3, 4) == (OK, [1, 3])
    assert o.pool_state()[0].tolist() == [1, 0, 1, 0, 0, 0] and o.protected_map().tolist() == [1, 0, 1, 0, 0, 0]


def test_demotion_event_precedes_the_loss_and_offloaded_claims_are_not_victims():
    o, pool, fill, ids = setup(8, [[0, 1], [2, 3], [4, 5]])
    assert o.offload([2])[0] == 0                                               # claim 2 holds no table any more
    st, got = o.make_room(4, 6)                                                 # 4 free + claim 1 (2) -> 6
    assert (st, got) == (OK, [1])
    assert o.claim_info(2)["state"] == 3                                        # offloaded: not a victim candidate
    # protection follows the claim through offload and restore
    assert o.protect([2], [1]) == 0 and not o.protected_map().any()
    assert o.restore([2])[0] == 0
    assert o.protected_map().tolist() == [1, 1, 0, 0, 0, 0, 0, 0]               # its new footprint (lowest free ids)
    st, got = o.make_room(5, 7)
    assert (st, got) == (CONFLICT, [2])
    ev = o.ev0 + list(o.outcomes())
    ok, why = V.validate(ev)
    assert ok, why
    i_dem = [i for i, e in enumerate(ev) if int(e["code"]) == 9][0]
    assert int(ev[i_dem]["claim_id"]) == 1 and int(ev[i_dem]["aux"]) == 2 and int(ev[i_dem]["arg"]) == 4


NBP = 8
SPEC = {1: [0, 1], 2: [2, 3], 3: [4]}


def test_no_call_sequence_ever_hands_out_or_alters_a_protected_block():
    """Brute force: three materialized claims on an 8-block pool, then a DFS over offload / restore / protect /
    unprotect / release / make_room(2, 4, 5, 7), three state-changing calls deep plus any fourth call.  After every call:
    the footprint of every protected claim the call did not name is still held by it, used, referenced and
    byte-identical; make_room never evicts a protected claim and a refusal evicts nobody; restore hands out free blocks
    only; no two claims hold the same block; every stream validates."""
    acts = [(op, c) for c in SPEC for op in ("offload", "restore", "protect", "unprotect", "release")]
    acts += [("room", need) for need in (2, 4, 5, 7)]

    def apply(o, act):
        op, c = act
        if op in ("protect", "unprotect"):
            return 0 if o.protect([c], [1 if op == "protect" else 0]) == 0 else -1
        if op == "room":
            return o.make_room(1000 + c, c)[0]
        return int(getattr(o, op)([c])[0])

    def state_of(o, c):
        info = o.claim_info(c)
        return info["state"] if info else None

    n_nodes = n_conflict = n_demoted = 0
    stack = [()]
    while stack:
        prefix = stack.pop()
        for act in acts:
            o, pool, fill, _ = setup(NBP, [SPEC[c] for c in sorted(SPEC)])
            view = pool.reshape(2 * L_, NBP, PAGE)
            flag = {c: 0 for c in SPEC}                    # the test's own record of the protect flags
            changed = False
            for a in prefix + (act,):
                states = {c: state_of(o, c) for c in SPEC}
                foot = {c: list(o.claim_blocks(c)) for c in SPEC if flag[c] and states[c] in (1, 2, 4)}
                held = {c: view[:, t, :].copy() for c, t in foot.items()}
                used0, ref0 = o.pool_state()
                flag0 = dict(flag)
                st = apply(o, a)
                if a[0] in ("protect", "unprotect") and st == 0:
                    flag[a[1]] = 1 if a[0] == "protect" else 0
                if a[0] == "release" and st == 0:
                    flag[a[1]] = 0
                used, ref = o.pool_state()
                for c, t in foot.items():                  # protected footprints of claims this call did not name
                    if a[0] != "room" and a[1] == c:
                        continue
                    assert state_of(o, c) == states[c] and list(o.claim_blocks(c)) == t, (prefix, act, a, c)
                    assert all(used[b] and ref[b] >= 1 for b in t)
                    assert np.array_equal(view[:, t, :], held[c])
                if a[0] == "room":
                    if st == 9:                            # refusal: nobody was evicted, no block changed hands
                        n_conflict += 1
                        assert {c: state_of(o, c) for c in SPEC} == states
                        assert np.array_equal(used, used0) and np.array_equal(ref, ref0)
                        assert any(flag[c] and states[c] in (1, 2, 4) for c in SPEC)
                    elif st == 0:
                        gone = [c for c in SPEC if states[c] != 6 and state_of(o, c) == 6]
                        assert not any(flag[c] for c in gone)                 # victims are unprotected claims only
                        n_demoted += len(gone)
                        assert int((used == 0).sum()) >= a[1]                 # the room was made
                    else:
                        assert st == 6 and np.array_equal(used, used0)
                if a[0] == "restore" and st == 0:
                    assert not used0[o.claim_blocks(a[1])].any()              # fresh blocks come from free ones only
                tables = [list(o.claim_blocks(c)) for c in SPEC if state_of(o, c) in (1, 2, 4)]
                flat = [b for t in tables for b in t]
                assert len(flat) == len(set(flat)) and int(ref.sum()) == len(flat) and all(used[b] for b in flat)
                assert np.array_equal(o.protected_map().nonzero()[0],
                                      sorted(b for c in SPEC if flag[c] and state_of(o, c) in (1, 2, 4) for b in o.claim_blocks(c)))
                changed = ({c: state_of(o, c) for c in SPEC} != states or flag != flag0 or not np.array_equal(used, used0))
            n_nodes += 1
            ok, why = V.validate(o.ev0 + list(o.outcomes()))
            assert ok, (prefix, act, why)
            if len(prefix) < 3 and changed:                # a call that changed nothing cannot matter to later calls
                stack.append(prefix + (act,))
            o.close()
    assert n_nodes > 3000 and n_conflict > 50 and n_demoted > 50
