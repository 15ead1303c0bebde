"""Event-stream validator -- ORACLE side, test infrastructure only.

The CPU restatement of the paper's artifact analyzer, which "supplies no runtime
behavior; it only checks order, claim match, and controls after the run"
(P:L331).  Input: a list of (seq, claim_id, code, aux, arg) tuples (or a numpy
record array with those fields).  Two harness-only marker codes may appear:
USE(C) = "the reuse request consumed the prefix" and REQUEST_FINISHED(C).

Accepted language per claim:
    ACCEPTED MATERIALIZED ( OFFLOADED RESTORE_REQUIRED
        ( RESTORED USE* | LOAD_FAILED RESTORATION_FAILED REFUSED ) )*
any prefix of it is valid; nothing but REQUEST_FINISHED follows REFUSED.
Rules and the passages that fix them:
  * seq strictly increasing;
  * no event names a claim before its ACCEPTED (post-hoc naming P:L257);
  * USE(C) while C is offloaded / restore-required is invalid: restore-after-use
    (P:L23);
  * REQUEST_FINISHED(C) between LOAD_FAILED and REFUSED is invalid: the outcome
    precedes terminal handling (path B row 8);
  * LOAD_FAILED / RESTORATION_FAILED / REFUSED without RESTORE_REQUIRED(C) in the
    same cycle is invalid: generic, unclaimed or wrong-claim failure (P:L25, P:L48,
    P:L463);
  * REFUSED.arg (blocking_claim_ids) must be [C], the refused claim itself.
Allocator-side protection (NEXT-3, DESIGN.md 12 / R23):
  * DEMOTED(C, arg = request id != 0) while C is resident (ACCEPTED / MATERIALIZED / RESTORED) is the ordered
    demotion of a victim before its blocks are lost (claim_demoted_before_loss); terminal like the other outcomes;
    DEMOTED after RESTORATION_FAILED keeps arg = 0;
  * CONFLICT_REFUSED(C, aux = REQ_FLAG | k, arg = request id): a resident claim C blocks an active request under hard
    protection; C stays as it is.  The k records of one refusal are consecutive and name k different claims.
"""
ACCEPTED, MATERIALIZED, OFFLOADED, RESTORE_REQUIRED, LOAD_FAILED, RESTORED, RESTORATION_FAILED, REFUSED = range(1, 9)
DEMOTED, EXPIRED = 9, 10          # NEXT-3: the other claim-scoped outcomes of a failed restoration
CONFLICT_REFUSED = 11             # NEXT-3: active_request_refused(blocking_claim_ids) under hard protection
USE, REQUEST_FINISHED = 100, 101
REQ_FLAG = 0x80000000             # REFUSED.aux of a request-level refusal: flag | size of blocking_claim_ids

# per-claim automaton states
_S0, _ACC, _MAT, _OFF, _RREQ, _LF, _RF, _REF, _RES, _FIN, _DEM, _EXP = range(12)

_NEXT = {
    (_S0, ACCEPTED): _ACC,
    (_ACC, MATERIALIZED): _MAT,
    (_MAT, OFFLOADED): _OFF,
    (_RES, OFFLOADED): _OFF,
    (_OFF, RESTORE_REQUIRED): _RREQ,
    (_RREQ, RESTORED): _RES,
    (_RREQ, LOAD_FAILED): _LF,
    (_LF, RESTORATION_FAILED): _RF,
    (_RF, REFUSED): _REF,
    (_RF, DEMOTED): _DEM,
    (_RF, EXPIRED): _EXP,
    (_MAT, USE): _MAT,
    (_RES, USE): _RES,
    (_REF, REQUEST_FINISHED): _FIN,
    (_DEM, REQUEST_FINISHED): _FIN,
    (_EXP, REQUEST_FINISHED): _FIN,
    (_ACC, REQUEST_FINISHED): _FIN,
    (_MAT, REQUEST_FINISHED): _FIN,
    (_RES, REQUEST_FINISHED): _FIN,
    # allocator-side protection: a resident victim is demoted before its blocks are lost; a protected resident claim
    # that blocks an active request is named and stays
    (_ACC, DEMOTED): _DEM, (_MAT, DEMOTED): _DEM, (_RES, DEMOTED): _DEM,
    (_ACC, CONFLICT_REFUSED): _ACC, (_MAT, CONFLICT_REFUSED): _MAT, (_RES, CONFLICT_REFUSED): _RES,
}


def _rows(events):
    out = []
    for ev in events:
        if hasattr(ev, "dtype") and ev.dtype.names:
            out.append((int(ev["seq"]), int(ev["claim_id"]), int(ev["code"]), int(ev["aux"]), int(ev["arg"])))
        else:
            s, c, code, aux, arg = ev
            out.append((int(s), int(c), int(code), int(aux), int(arg)))
    return out


def _scan(events):
    """The analyzer loop: (ok, index of the first violation or -1, reason).

    Request-level refusals (NEXT-3; P:L87 blocking_claim_ids, "smear blocking ids across claims ...
    fails closed"): a reuse request naming several claims is refused once, by a run of consecutive
    REFUSED records with the same arg (request id) and aux = REQ_FLAG | k, one per blocking claim.  The run must
    name exactly the k claims whose restoration failed and is still unanswered (state RF) -- neither a claim
    that did not fail (the automaton rejects it) nor fewer than all that did (k must equal the pending count),
    and nothing may interrupt the run."""
    state = {}
    last_seq = None
    pending = 0                     # claims in state RF: failed, outcome not yet emitted
    group = None                    # [arg, aux, records still to come]
    cgroup = None                   # the same for a CONFLICT_REFUSED run, plus the claims it has named
    cdone = None                    # (arg, aux) of the CONFLICT_REFUSED run that ended with the previous record
    for i, (seq, cid, code, aux, arg) in enumerate(_rows(events)):
        if last_seq is not None and seq <= last_seq:
            return False, i, "seq not strictly increasing at %d" % seq
        last_seq = seq
        if cid == 0:
            return False, i, "event names no claim (unclaimed) at seq %d" % seq
        if group is not None and not (code == REFUSED and arg == group[0] and aux == group[1]):
            return False, i, "blocking_claim_ids run of request %#x interrupted (seq %d)" % (group[0], seq)
        if cgroup is not None and not (code == CONFLICT_REFUSED and arg == cgroup[0] and aux == cgroup[1]):
            return False, i, "blocking_claim_ids run of request %#x interrupted (seq %d)" % (cgroup[0], seq)
        s = state.get(cid, _S0)
        nxt = _NEXT.get((s, code))
        if code == DEMOTED and nxt is not None and (arg == 0) != (s == _RF):
            nxt = None                                  # arg = 0 after a failed restoration, = request id for a victim
        if code == CONFLICT_REFUSED and nxt is not None:
            k = aux & ~REQ_FLAG
            if not (aux & REQ_FLAG) or k == 0 or arg == 0:
                nxt = None
            elif cgroup is None and cdone == (arg, aux):
                return False, i, "request %#x: more blocking_claim_ids records than announced (seq %d)" % (arg, seq)
            elif cgroup is None:
                cgroup = [arg, aux, k, set()]
            if nxt is not None:
                if cid in cgroup[3]:
                    return False, i, "request %#x: blocking claim %#x named twice (seq %d)" % (arg, cid, seq)
                cgroup[3].add(cid)
                cgroup[2] -= 1
                if cgroup[2] == 0:
                    cgroup = None
                    cdone = (arg, aux)
                    state[cid] = nxt
                    continue
        cdone = None
        if nxt is None:
            return False, i, "claim %#x: code %d not allowed in state %d (seq %d)" % (cid, code, s, seq)
        if code == RESTORATION_FAILED:
            pending += 1
        elif code == EXPIRED or (code == DEMOTED and s == _RF):
            pending -= 1
        elif code == REFUSED:
            if aux & REQ_FLAG:
                if group is None:
                    k = aux & ~REQ_FLAG
                    if k == 0 or k != pending:
                        return False, i, "request %#x: blocking_claim_ids is not the exact failed subset (seq %d)" % (arg, seq)
                    group = [arg, aux, k]
                group[2] -= 1
                if group[2] == 0:
                    group = None
            elif arg != cid or aux != 1:
                return False, i, "claim %#x: blocking_claim_ids is not [C] (seq %d)" % (cid, seq)
            pending -= 1
        state[cid] = nxt
    return True, -1, "ok"


def validate(events):
    """Returns (ok, reason).  ok is True iff the whole stream is in the accepted language."""
    ok, _, why = _scan(events)
    return ok, why


FAILURE_ORDER = [ACCEPTED, MATERIALIZED, OFFLOADED, RESTORE_REQUIRED, LOAD_FAILED, RESTORATION_FAILED, REFUSED]
SUCCESS_ORDER = [ACCEPTED, MATERIALIZED, OFFLOADED, RESTORE_REQUIRED, RESTORED]


def codes_of(events, cid):
    return [code for _, c, code, _, _ in _rows(events) if c == cid]


def failure_outcome_gate(events, cid):
    """Same-claim failure outcome gate: the stream is valid and C's own subsequence
    ends with the exact seven-step order printed at P:L27."""
    ok, _ = validate(events)
    codes = [c for c in codes_of(events, cid) if c not in (USE, REQUEST_FINISHED)]
    if not ok or len(codes) < 7:
        return False
    tail = codes[-7:] if len(codes) == 7 else codes[:2] + codes[-5:]
    return tail == FAILURE_ORDER


def observation_gate(events, cid):
    """Positive observation gate (path A): C's subsequence ends with
    OFFLOADED RESTORE_REQUIRED RESTORED and no failure record names C."""
    ok, _ = validate(events)
    codes = [c for c in codes_of(events, cid) if c not in (USE, REQUEST_FINISHED)]
    return bool(ok and len(codes) >= 5 and codes[:2] == SUCCESS_ORDER[:2] and codes[-3:] == SUCCESS_ORDER[-3:]
                and LOAD_FAILED not in codes and REFUSED not in codes)


def validate_index(events):
    """validate() with the stream position of the first violation: (True, -1) or (False, index)."""
    ok, i, _ = _scan(events)
    return ok, i
