"""Pins that fix the oracle against the paper and the mathematics by brute force on tiny inputs (-m "not gpu").

(i)   predicate: leading-prefix-at-least-N (hit=448 served P:L364-367) by its token-level definition,
      exhaustive over every fill vector of a 3-block claim with BS = 4, every P in 9..12 and every N in 1..P; plus
      M = N-1, N, N+1 at BS = 16.  A predicate that counts materialized tokens instead of the LEADING run fails here.
(ii)  validator: the per-claim language of SURVEY 8(c).4 restated as a
      regular expression; the validator must agree with it on every (reachable state, next code) pair, on all 7! and
      5! permutations of the two paths, and on all interleavings of two claims (accepted iff order-preserving).
(iii) call sequences: every sequence of accept / materialize / offload / restore (fault armed or not) / release calls
      over 2 claims on an 8-block pool, to depth 7 (6 state-changing calls, then any call): every emitted stream validates, every
      illegal call emits nothing and changes nothing, allocator invariants hold after every call.
(iv)  allocator (DESIGN R6/R7): a restore receives sorted(free)[:nb] per claim in batch order, after arbitrary
      mark_used / mark_free patterns; sum(ref) = live table entries; a served prefix, then NO_FREE_BLOCKS.
"""
import itertools

import numpy as np
import pytest
import regex

from oracle import rco, validator as V

# a geometry with BS = 4 whose page is still a multiple of 4096 bytes: 4 tokens x 4 heads x 128 dims x 2 bytes
L_, H_, D_, E_, BS4 = 1, 4, 128, 2, 4
PAGE = BS4 * H_ * D_ * E_
BLK = 2 * L_ * PAGE


def small_oracle(nb_pool, bs=BS4, seed=0, host=1 << 40):
    h = H_ if bs == 4 else 1
    pool = np.random.default_rng(seed).integers(0, 256, 2 * L_ * nb_pool * bs * h * D_ * E_, dtype=np.uint8)
    fill = np.zeros(nb_pool, np.uint8)
    o = rco.Oracle(L_, h, D_, E_, bs, nb_pool, pool, fill, host)
    return o, pool, fill


# ---- (i) predicate ---------------------------------------------------------------------------------------------------
def leading_run(P, bs, bt, fill):
    """mat(t) := (t mod BS) < fill[bt[t div BS]];  M := the first t that is not materialized, else P."""
    return next((t for t in range(P) if not (t % bs) < fill[bt[t // bs]]), P)


def test_predicate_exhaustive_over_all_fill_vectors_bs4():
    o, pool, fill = small_oracle(8)
    bt = [5, 2, 7]                                         # a permuted table: physical order != logical order
    o.mark_used(bt)
    cid = 0
    n_true = n_false = n_sum_differs = 0
    for P in (9, 10, 11, 12):                              # last block holds 1..4 tokens
        for f in itertools.product(range(BS4 + 1), repeat=3):     # 125 fill vectors, incl. holes and fill > cap
            fill[:] = 0
            fill[bt] = f
            M = leading_run(P, BS4, bt, fill)
            total = sum(min(f[i], min(BS4, P - i * BS4)) for i in range(3))   # what a summing predicate would see
            n_sum_differs += total != M
            for N in range(1, P + 1):
                cid += 1
                o.mark_used(bt)                            # release hands the blocks back to the free list
                assert o.accept([cid], [P], [N], [0, 3], bt)[0] == 0
                st = int(o.materialize([cid])[0])
                info = o.claim_info(cid)
                if M >= N:                                 # ">=": a hit of exactly N tokens is served
                    assert st == 0 and info["M"] == M and info["nb"] == -(-M // BS4) and info["state"] == 2
                    n_true += 1
                else:                                      # no event, claim stays ACCEPTED
                    assert st == 1 and info["state"] == 1 and info["M"] == 0
                    n_false += 1
                o.release([cid])
    ev = o.outcomes()
    assert sum(1 for e in ev if int(e["code"]) == 2) == n_true and len(ev) == cid + n_true
    assert n_true > 1000 and n_false > 1000
    assert n_sum_differs > 150                             # the inputs do separate "leading run" from "count"


@pytest.mark.parametrize("M", [447, 448, 449, 0, 1, 15, 16, 17, 460])
def test_predicate_boundary_at_448_bs16(M):
    o, pool, fill = small_oracle(40, bs=16)
    P, N = 460, 448
    bt = list(np.random.default_rng(3).permutation(40)[:29])
    o.mark_used(bt)
    for i, b in enumerate(bt):                             # M leading tokens, then a hole, then full blocks again
        fill[b] = min(16, max(0, M - i * 16))
    for i in range(M // 16 + 1, 29):
        fill[bt[i]] = 16
    assert leading_run(P, 16, bt, fill) == M
    assert o.accept([9], [P], [N], [0, 29], bt)[0] == 0
    st = int(o.materialize([9])[0])
    assert st == (0 if M >= 448 else 1)
    if M >= 448:
        assert o.claim_info(9)["M"] == M and o.claim_info(9)["nb"] == -(-M // 16)
        assert [int(e["aux"]) for e in o.outcomes() if int(e["code"]) == 2] == [M]


# ---- (ii) validator ----------------------------------------------------------------------------------------------------
# one letter per code; the per-claim language of SURVEY 8(c).4 (with DEMOTED / EXPIRED of NEXT-3 as the other outcomes):
#   A M U* ( O R S U* )* ( O R L F (X|D|E) )? Z?   or   A Z        -- any prefix of such a word is valid
LET = {V.ACCEPTED: "A", V.MATERIALIZED: "M", V.OFFLOADED: "O", V.RESTORE_REQUIRED: "R", V.RESTORED: "S",
       V.LOAD_FAILED: "L", V.RESTORATION_FAILED: "F", V.REFUSED: "X", V.DEMOTED: "D", V.EXPIRED: "E", V.USE: "U",
       V.REQUEST_FINISHED: "Z"}
CODE = {v: k for k, v in LET.items()}
LANG = regex.compile(r"A(?:Z|MU*(?:ORSU*)*(?:ORLF[XDE])?Z?)")


def in_language(word):
    return word == "" or LANG.fullmatch(word, partial=True) is not None


def stream(words):
    """Event list from [(claim id, letter), ...] in stream order; REFUSED carries blocking_claim_ids = [C]."""
    return [(i, c, CODE[ch], 1 if ch == "X" else 0, c if ch == "X" else 0) for i, (c, ch) in enumerate(words)]


def test_validator_agrees_with_the_grammar_on_every_state_and_code():
    # all valid words up to length 11 (branching is small), each extended by every one of the 12 codes
    frontier, seen, checked, rejected = [""], set(), 0, 0
    while frontier:
        w = frontier.pop()
        for ch in LET.values():
            x = w + ch
            want = in_language(x)
            ok, idx = V.validate_index(stream([(7, c) for c in x]))
            assert ok == want, (x, ok, want)
            if not want:
                assert idx == len(w)                       # the first violation is the appended record
                rejected += 1
            elif len(x) < 11 and x not in seen:
                seen.add(x)
                frontier.append(x)
            checked += 1
    assert checked > 1800 and rejected > 1400 and len(seen) > 150
    # the forbidden edges the paper names, one by one
    for bad, why in [("AMORLFZ", "terminal handling before the outcome, P:L380"),
                     ("AMORLZ", "terminal handling before the outcome, P:L380"),
                     ("AMOU", "restore-after-use, P:L23 / P:L448"), ("AMORU", "use while restore-required"),
                     ("AO", "offloaded before materialized"), ("M", "lifecycle event before accept, P:L333"),
                     ("AMORLFS", "fallback recompute after a failed load, P:L492"),
                     ("AML", "generic failure without restore-required, P:L48 / P:L493"),
                     ("AMOL", "failure without restore-required"), ("AMORLFXO", "refused is terminal"),
                     ("AMORLFXX", "refused twice"), ("AMORSS", "restored twice"), ("AA", "duplicate accept, P:L199")]:
        assert not V.validate(stream([(7, c) for c in bad]))[0], (bad, why)


@pytest.mark.parametrize("path", ["AMORLFX", "AMORS"])
def test_only_the_papers_order_of_each_path_is_accepted(path):
    # P:L27 (seven steps) and path A: of all permutations only the printed order passes
    n_ok = 0
    for perm in itertools.permutations(path):
        ok, _ = V.validate(stream([(3, c) for c in perm]))
        assert ok == ("".join(perm) == path)
        n_ok += ok
    assert n_ok == 1
    ev = stream([(3, c) for c in path])
    assert V.failure_outcome_gate(ev, 3) == (path == "AMORLFX") and V.observation_gate(ev, 3) == (path == "AMORS")


def test_two_claim_interleavings_accepted_iff_order_preserving():
    a, b = "AMORLFX", "AMORS"
    rng = np.random.default_rng(4)
    n = 0
    for pos in itertools.combinations(range(12), 5):       # all 792 interleavings: positions of claim 2's events
        ia, ib = iter(a), iter(b)
        words = [(2, next(ib)) if i in pos else (1, next(ia)) for i in range(12)]
        ev = stream(words)
        assert V.validate(ev)[0]
        assert V.failure_outcome_gate(ev, 1) and V.observation_gate(ev, 2)        # target-only attribution
        assert not V.failure_outcome_gate(ev, 2) and not V.observation_gate(ev, 1)
        # any exchange of two events of one claim breaks that claim's order -> rejected
        who = 1 if rng.random() < 0.5 else 2
        idx = [i for i, (c, _) in enumerate(words) if c == who]
        i, j = sorted(rng.choice(len(idx), 2, replace=False))
        sw = list(words)
        sw[idx[i]], sw[idx[j]] = words[idx[j]], words[idx[i]]
        assert not V.validate(stream(sw))[0]
        n += 1
    assert n == 792
    for pos in itertools.combinations(range(14), 7):       # two failure paths: all 3432 interleavings
        ia, ib = iter(a), iter(a)
        ev = stream([(2, next(ib)) if i in pos else (1, next(ia)) for i in range(14)])
        assert V.validate(ev)[0] and V.failure_outcome_gate(ev, 1) and V.failure_outcome_gate(ev, 2)
    # wrong-claim: claim 2's failure records carry claim 1's id
    ev = stream([(1, c) for c in "AMOR"] + [(2, c) for c in "AMOR"] + [(1, "L"), (1, "F"), (1, "X"), (1, "L")])
    assert not V.validate(ev)[0]
    ev = stream([(1, c) for c in "AMORLF"])
    ev.append((6, 1, V.REFUSED, 1, 2))                     # blocking_claim_ids names another claim
    assert not V.validate(ev)[0]
    ev[-1] = (6, 1, V.REFUSED, 2, 1)                       # |blocking_claim_ids| != 1 in the per-claim form
    assert not V.validate(ev)[0]
    ev[-1] = (5, 1, V.REFUSED, 1, 1)                       # seq not strictly increasing
    assert not V.validate(ev)[0]
    ev[-1] = (6, 1, V.REFUSED, 1, 1)
    assert V.validate(ev)[0]


# ---- (iii) enumerated call sequences -----------------------------------------------------------------------------------
NBP = 8
CLAIMS = {11: dict(P=8, N=5, bt=[6, 1]), 22: dict(P=6, N=4, bt=[3, 4])}
ACTIONS = [(op, c) for c in CLAIMS for op in ("accept", "materialize", "offload", "restore", "restore_xfer",
                                              "restore_flip", "release")]


def fresh():
    o, pool, fill = small_oracle(NBP, seed=1)
    o.mark_used([1, 3, 4, 6])
    fill[[1, 3, 4, 6]] = 4
    return o, pool, fill


def apply(o, act):
    op, c = act
    if op == "accept":
        s = CLAIMS[c]
        return int(o.accept([c], [s["P"]], [s["N"]], [0, len(s["bt"])], s["bt"])[0])
    if op.startswith("restore"):
        o.set_faults({"restore": [], "restore_xfer": [(c, 1, 0)], "restore_flip": [(c, 2, 12345)]}[op])
        st = int(o.restore([c])[0])
        o.set_faults([])
        return st
    return int(getattr(o, op)([c])[0])


def snapshot(o, pool, fill):
    used, ref = o.pool_state()
    live = [b for b in range(NBP) if used[b]]
    view = pool.reshape(2 * L_, NBP, PAGE)
    return (used.tobytes(), ref.tobytes(), fill[live].tobytes(), view[:, live, :].tobytes(),
            tuple(sorted((c, tuple(sorted(o.claim_info(c).items()))) for c in CLAIMS if o.claim_info(c))),
            o.stats()["host_used"])


def check_invariants(o):
    used, ref = o.pool_state()
    tables = [o.claim_blocks(c) for c in CLAIMS if o.claim_info(c) is not None]
    assert int(ref.sum()) == sum(len(t) for t in tables)                       # sum(ref) = live table entries
    assert all(used[b] for t in tables for b in t)
    flat = [int(b) for t in tables for b in t]
    assert len(flat) == len(set(flat))                                         # these claims never share a block
    assert int((used == 0).sum()) + int((used == 1).sum()) == NBP


def test_every_call_sequence_emits_only_valid_streams_and_illegal_calls_emit_nothing():
    """DFS over the state-changing calls to depth 6 (8078 calls in all); at every node all 14 actions are tried.  A call that returns
    a status other than OK / RESTORE_FAILED must leave the event count, the allocator, fill, the live pool bytes,
    every claim and the host store untouched (it cannot change what later calls see, so it need not be explored
    further).  Every stream produced must be in the validator's language, and a restore with an armed fault must end
    in the seven-step order."""
    nodes = illegal = legal = failures = 0
    terminal_states = set()
    stack = [()]
    while stack:
        prefix = stack.pop()
        for act in ACTIONS:
            o, pool, fill = fresh()
            for a in prefix:
                apply(o, a)
            n0, snap0 = o.stats()["n_events"], snapshot(o, pool, fill)
            st = apply(o, act)
            nodes += 1
            if st in (0, 8) :
                legal += 1
                check_invariants(o)
                ev = o.outcomes()
                ok, why = V.validate(ev)
                assert ok, (prefix, act, why)
                if act[0] == "release":
                    assert o.stats()["n_events"] == n0 and o.claim_info(act[1]) is None     # emits nothing
                elif st == 8:
                    failures += 1
                    assert act[0] in ("restore_xfer", "restore_flip")
                    codes = [int(e["code"]) for e in ev if int(e["claim_id"]) == act[1]]
                    assert codes[-4:] == [4, 5, 7, 8] and int(ev[-1]["arg"]) == act[1]     # P:L27 tail, [C]
                    assert o.claim_info(act[1])["state"] == 5
                    terminal_states.add(act[1])
                else:
                    assert o.stats()["n_events"] == n0 + (2 if act[0].startswith("restore") else 1)
                    if act[0].startswith("restore"):
                        assert act[0] == "restore"         # an armed same-claim fault never yields RESTORED
                if len(prefix) < 6:
                    stack.append(prefix + (act,))
            else:
                illegal += 1
                assert o.stats()["n_events"] == n0, (prefix, act, st)          # no claim outcome
                assert snapshot(o, pool, fill) == snap0, (prefix, act, st)
            o.close()
    assert nodes > 5000 and illegal > 3000 and legal > 1000 and failures > 100 and terminal_states == {11, 22}


# ---- (iv) allocator -----------------------------------------------------------------------------------------------------
def test_restore_takes_the_lowest_free_ids_in_batch_order():
    rng = np.random.default_rng(12)
    for trial in range(40):
        nbp = 24
        o, pool, fill = small_oracle(nbp, seed=trial)
        perm = [int(b) for b in rng.permutation(nbp)]
        specs, cur = [], 0
        for cid in (1, 2, 3):
            nt = int(rng.integers(1, 5))
            specs.append((cid, 4 * nt - int(rng.integers(0, 4)), perm[cur:cur + nt]))
            cur += nt
        o.mark_used(perm[:cur])
        fill[perm[:cur]] = 4
        for cid, P, bt in specs:
            assert o.accept([cid], [P], [1], [0, len(bt)], bt)[0] == 0
        ids = [s[0] for s in specs]
        assert not o.materialize(ids).any() and not o.offload(ids).any()
        used, ref = o.pool_state()
        assert not used.any() and not ref.any()                                # offload dropped every reference (R5)
        # an arbitrary occupancy pattern, built by marking used and freeing again
        occ = rng.random(nbp) < rng.uniform(0.2, 0.8)
        o.mark_used(np.nonzero(occ)[0])
        back = np.nonzero(occ & (rng.random(nbp) < 0.3))[0]
        o.mark_free(back)
        occ[back] = False
        free = [b for b in range(nbp) if not occ[b]]
        order = [int(x) for x in rng.permutation(3)]                            # batch order != id order
        batch = [ids[k] for k in order]
        nbs = [o.claim_info(c)["nb"] for c in batch]
        st = o.restore(batch)
        take, served = 0, []
        for c, nb in zip(batch, nbs):                                          # prefix rule (R7): served while the sum fits
            if take + nb > len(free):
                break
            served.append(c)
            take += nb
        assert list(st) == [0] * len(served) + [6] * (3 - len(served))
        cursor = 0
        for c, nb in zip(batch, nbs):
            if c in served:
                assert list(o.claim_blocks(c)) == free[cursor:cursor + nb]      # lowest free ids, ascending (R6)
                cursor += nb
            else:
                assert o.claim_info(c)["state"] == 3 and len(o.claim_blocks(c)) == 0
        used, ref = o.pool_state()
        assert int(ref.sum()) == cursor                                        # sum(ref) = live table entries
        assert int(used.sum()) == int(occ.sum()) + cursor and int((used == 0).sum()) == nbp - int(used.sum())
        assert all(ref[b] == 1 for c in served for b in o.claim_blocks(c))
        o.close()


def test_shared_blocks_are_freed_only_by_their_last_reference():
    o, pool, fill = small_oracle(8)
    o.mark_used([0, 1, 2, 3])
    fill[:4] = 4
    assert o.accept([1, 2], [8, 8], [1, 1], [0, 2, 4], [0, 1, 0, 2]).tolist() == [0, 0]   # block 0 shared between claims
    _, ref = o.pool_state()
    assert ref[:4].tolist() == [2, 1, 1, 0]
    assert not o.materialize([1, 2]).any()
    assert o.offload([1])[0] == 0
    used, ref = o.pool_state()
    assert used[:4].tolist() == [1, 0, 1, 1] and ref[:4].tolist() == [1, 0, 1, 0]         # 3 was marked, never claimed
    assert o.offload([2])[0] == 0
    used, ref = o.pool_state()
    assert used[:4].tolist() == [0, 0, 0, 1] and not ref.any()
