"""Synthetic event traces and their control-class mutations: inputs of the trace validator (NEXT-1 / NEXT-3).

Test infrastructure (inputs only; the grammar they are checked against lives in oracle/validator.py and in the CUDA
validator).  bench.py's trace_validator leg draws its 200k-claim stream from make_trace.
"""
import numpy as np

SEED0 = 260601387

# ---- synthetic event traces (inputs of the trace validator, NEXT-1) -----------------------------------
TRACE_DTYPE = np.dtype([("seq", "<u8"), ("claim_id", "<u8"), ("code", "<u4"), ("aux", "<u4"), ("arg", "<u8")])
T_USE, T_FIN = 100, 101
TRACE_MUTATIONS = ["wrong_claim", "unclaimed", "restore_after_use", "finish_before_refused", "drop_restore_required",
                   "swap_adjacent", "bad_blocking_ids", "seq_not_increasing", "generic_failure", "fallback_recompute"]


def make_trace(n_claims, seed=0, fail_frac=0.1, cycles=(1, 3), markers=True):
    """A valid interleaved stream: each claim runs ACCEPTED, MATERIALIZED, then 1..3 offload/restore cycles;
    a fraction end in the failure path (the seven steps of P:L27); optional USE / REQUEST_FINISHED markers.
    Events of different claims are interleaved at random, per-claim order kept.  Vectorised (10^6 claims ok)."""
    rng = np.random.default_rng(SEED0 + 5000 + seed)
    ids = rng.integers(1, 1 << 62, n_claims, dtype=np.uint64) * np.uint64(2) + np.uint64(1)
    ids = np.unique(ids)
    rng.shuffle(ids)
    n = ids.size
    ncyc = rng.integers(cycles[0], cycles[1] + 1, n)
    fail = rng.random(n) < fail_frac
    use = (rng.random(n) < 0.3) & ~fail & markers
    fin = (rng.random(n) < 0.3) & markers
    cols = []                                              # per-claim code sequences as padded columns
    L = 2 + 3 * cycles[1] + 2 + 2
    seqs = np.zeros((n, L), np.uint32)
    ln = np.zeros(n, np.int64)

    def push(mask, code):
        idx = np.nonzero(mask)[0]
        seqs[idx, ln[idx]] = code
        ln[idx] += 1
    allm = np.ones(n, bool)
    push(allm, 1); push(allm, 2)
    for cyc in range(cycles[1]):
        act = ncyc > cyc
        last = ncyc == cyc + 1
        push(act, 3); push(act, 4)
        push(act & ~(last & fail), 6)
        push(act & last & fail, 5); push(act & last & fail, 7); push(act & last & fail, 8)
    push(use, T_USE)
    push(fin, T_FIN)
    total = int(ln.sum())
    owner = np.repeat(np.arange(n), ln)
    within = np.arange(total) - np.repeat(np.cumsum(ln) - ln, ln)
    t = rng.random(total)
    # per-claim sorted times keep the claim's own order
    order_in = np.lexsort((t, owner))
    t_sorted = np.empty(total)
    t_sorted[np.arange(total)] = t[order_in]
    glob = np.argsort(t_sorted, kind="stable")
    ev = np.zeros(total, TRACE_DTYPE)
    code = seqs[owner, within]
    ev["claim_id"] = ids[owner][glob]
    ev["code"] = code[glob]
    ev["seq"] = np.arange(total, dtype=np.uint64) * np.uint64(3) + np.uint64(7)
    ref = ev["code"] == 8
    ev["aux"][ref] = 1
    ev["arg"][ref] = ev["claim_id"][ref]
    return ev


def mutate_trace(ev, kind, seed=0):
    """One control-class mutation applied to a valid stream; returns a new array."""
    rng = np.random.default_rng(SEED0 + 6000 + seed)
    ev = ev.copy()
    code, cid = ev["code"], ev["claim_id"]

    def pick(mask):
        idx = np.nonzero(mask)[0]
        return int(idx[rng.integers(0, idx.size)]) if idx.size else None

    def insert(pos, c, code_):
        rec = np.zeros(1, TRACE_DTYPE)
        rec["claim_id"], rec["code"] = c, code_
        out = np.concatenate([ev[:pos], rec, ev[pos:]])
        out["seq"] = np.arange(out.size, dtype=np.uint64) + np.uint64(1)
        return out
    if kind == "wrong_claim":                    # a failure record attributed to another claim
        i = pick(code == 5)
        other = cid[pick(cid != cid[i])]
        ev["claim_id"][i] = other
    elif kind == "unclaimed":
        ev["claim_id"][pick(code == 5)] = 0
    elif kind == "restore_after_use":            # USE(C) while C is offloaded
        i = pick(code == 3)
        return insert(i + 1, cid[i], T_USE)
    elif kind == "finish_before_refused":        # terminal handling before the outcome
        i = pick(code == 5)
        return insert(i + 1, cid[i], T_FIN)
    elif kind == "drop_restore_required":
        i = pick(code == 4)
        return np.delete(ev, i)
    elif kind == "swap_adjacent":                # two consecutive events of one claim exchanged
        i = pick(code == 3)
        j = i + 1 + int(np.nonzero(cid[i + 1:] == cid[i])[0][0])
        tmp = ev[["code", "aux", "arg"]][i].copy()
        for f in ("code", "aux", "arg"):
            a, b = ev[f][i], ev[f][j]
            ev[f][i], ev[f][j] = b, a
    elif kind == "bad_blocking_ids":             # blocking_claim_ids smeared onto another claim
        i = pick(code == 8)
        ev["arg"][i] = cid[pick(cid != cid[i])]
    elif kind == "seq_not_increasing":
        i = int(rng.integers(1, ev.size))
        ev["seq"][i] = ev["seq"][i - 1]
    elif kind == "generic_failure":              # failure records for a claim that was never restore-required
        i = pick(code == 2)
        return insert(i + 1, cid[i], 5)
    elif kind == "fallback_recompute":           # RESTORED after a failed load
        i = pick(code == 7)
        ev["code"][i] = 6
    else:
        raise ValueError(kind)
    return ev


REQ_FLAG = 0x80000000
REQUEST_MUTATIONS = ["smeared_ids", "short_subset", "dropped_record", "extra_record", "other_request_id", "interrupted_run",
                     "zero_subset", "early_finish"]


def make_request_trace(n_requests, seed=0):
    """Valid streams with multi-claim reuse requests (NEXT-3): every request names 2..5 offloaded claims; some fail
    and are refused (request-level run), demoted or expired.  Returns (events, runs) where runs lists, per refused
    request, the stream positions of its REFUSED records."""
    rng = np.random.default_rng(SEED0 + 8000 + seed)
    rows, hist, runs = [], [], []
    next_id = 1
    for r in range(n_requests):
        m = int(rng.integers(2, 6))
        cids = [int(next_id + 2 * j + 1) * 1000003 for j in range(m)]
        next_id += 2 * m
        for c in cids:
            hist.append([(c, 1, 0, 0), (c, 2, 0, 0), (c, 3, 0, 0)])
        req = 10 ** 12 + r
        blocking = []
        block = []
        for c in cids:
            block.append((c, 4, 0, 0))
            u = rng.random()
            if u < 0.55:
                block.append((c, 6, 0, 0))
            else:
                block += [(c, 5, 0, 0), (c, 7, 0, 0)]
                if u < 0.65:
                    block.append((c, 9, 0, 0))
                elif u < 0.75:
                    block.append((c, 10, 0, 0))
                else:
                    blocking.append(c)
        grp = [(c, 8, REQ_FLAG | len(blocking), req) for c in blocking]
        rows.append((block, grp))
    # histories interleaved at random (per-claim order kept), then the request blocks one after another
    order = np.repeat(np.arange(len(hist)), 3)
    rng.shuffle(order)
    it = [iter(h) for h in hist]
    flat = [next(it[k]) for k in order]
    for block, grp in rows:
        flat += block
        if grp:
            runs.append(list(range(len(flat), len(flat) + len(grp))))
        flat += grp
    ev = np.zeros(len(flat), TRACE_DTYPE)
    for i, (c, code, aux, arg) in enumerate(flat):
        ev[i] = (2 * i + 1, c, code, aux, arg)
    return ev, runs


def mutate_request_trace(ev, runs, kind, seed=0):
    rng = np.random.default_rng(SEED0 + 9000 + seed)
    ev = ev.copy()
    big = [r for r in runs if len(r) >= 2] or runs
    run = big[int(rng.integers(0, len(big)))]
    req = ev["arg"][run[0]]

    def reseq(a):
        a["seq"] = np.arange(a.size, dtype=np.uint64) + np.uint64(1)
        return a
    if kind == "smeared_ids":                    # names a claim of the request that restored fine
        start = run[0]
        i = start - 1
        while i >= 0 and ev["code"][i] != 6:
            i -= 1
        ev["claim_id"][run[-1]] = ev["claim_id"][i]
    elif kind == "short_subset":                 # fewer ids than claims that failed
        if len(run) >= 2:
            ev["aux"][run] = REQ_FLAG | (len(run) - 1)
            return reseq(np.delete(ev, run[-1]))
        ev["aux"][run] = REQ_FLAG | 2
    elif kind == "dropped_record":
        return reseq(np.delete(ev, run[0])) if len(run) >= 2 else reseq(np.delete(ev, run[0] - 1))
    elif kind == "extra_record":
        return reseq(np.concatenate([ev[:run[-1] + 1], ev[run[-1]:run[-1] + 1], ev[run[-1] + 1:]]))
    elif kind == "other_request_id":
        ev["arg"][run[-1]] = req + np.uint64(12345)
    elif kind == "interrupted_run":              # something else between the records of one run
        if len(run) < 2:
            ev["aux"][run] = REQ_FLAG | 2
        else:
            i = run[0] - 1
            while ev["code"][i] not in (6, 9, 10, 3):
                i -= 1
            rec = np.zeros(1, TRACE_DTYPE)
            rec["claim_id"], rec["code"] = ev["claim_id"][i], T_FIN
            return reseq(np.concatenate([ev[:run[1]], rec, ev[run[1]:]]))
    elif kind == "zero_subset":
        ev["aux"][run] = REQ_FLAG
    elif kind == "early_finish":                 # terminal handling before the request's outcome
        rec = np.zeros(1, TRACE_DTYPE)
        rec["claim_id"], rec["code"] = ev["claim_id"][run[0]], T_FIN
        return reseq(np.concatenate([ev[:run[0]], rec, ev[run[0]:]]))
    else:
        raise ValueError(kind)
    return ev


# ---- allocator-side protection (NEXT-3): victim demotions and protected-conflict refusals ------------------------------
T_CONFLICT = 11
PRESSURE_MUTATIONS = ["event_after_victim_demotion", "victim_demotion_without_request", "short_run", "interrupted_conflict_run",
                      "conflict_names_offloaded_claim", "claim_named_twice", "extra_conflict_record", "conflict_without_flag",
                      "failed_restore_demotion_with_request"]


def make_pressure_trace(n_rounds, seed=0):
    """Valid streams of an allocator under pressure: resident claims, rounds of make_room outcomes -- a prefix of
    unprotected claims demoted (DEMOTED, arg = request id) or a refusal run of k CONFLICT_REFUSED records naming k
    resident protected claims -- mixed with offload / restore cycles (some failing, some demoted with arg = 0).
    Returns (events, runs): runs = stream positions of each refusal run."""
    rng = np.random.default_rng(SEED0 + 9500 + seed)
    flat, runs = [], []
    nid = [1]

    def new_claim():
        c = nid[0] * 2654435761 % (1 << 61) + 17
        nid[0] += 1
        flat.append((c, 1, 448, 500)); flat.append((c, 2, 500, 0))
        return c
    for r in range(n_rounds):
        req = 5000 + r
        res = [new_claim() for _ in range(int(rng.integers(3, 9)))]          # resident claims of this round
        prot = [c for c in res if rng.random() < 0.4]
        unprot = [c for c in res if c not in prot]
        cyc = [c for c in res if rng.random() < 0.3]                          # some go through an offload cycle first
        for c in cyc:
            flat.append((c, 3, 30, 0)); flat.append((c, 4, 500, 0))
            u = rng.random()
            if u < 0.7:
                flat.append((c, 6, 30, 0))
            else:
                flat += [(c, 5, 0, 0), (c, 7, 0, 0)]
                flat.append((c, 9, 0, 0) if u < 0.85 else (c, 8, 1, c))
                res.remove(c)
                (prot if c in prot else unprot).remove(c)
        if unprot and rng.random() < 0.6:
            m = int(rng.integers(1, len(unprot) + 1))
            for c in unprot[:m]:
                flat.append((c, 9, int(rng.integers(1, 40)), req))
        elif prot:
            k = int(rng.integers(1, len(prot) + 1))
            runs.append(list(range(len(flat), len(flat) + k)))
            for c in prot[:k]:
                flat.append((c, T_CONFLICT, REQ_FLAG | k, req))
            if rng.random() < 0.5:                                           # the blockers live on
                flat.append((prot[0], 3, 30, 0))
    ev = np.zeros(len(flat), TRACE_DTYPE)
    for i, (c, code, aux, arg) in enumerate(flat):
        ev[i] = (3 * i + 2, c, code, aux, arg)
    return ev, runs


def mutate_pressure_trace(ev, runs, kind, seed=0):
    rng = np.random.default_rng(SEED0 + 9600 + seed)
    ev = ev.copy()
    big = [r for r in runs if len(r) >= 2] or runs
    run = big[int(rng.integers(0, len(big)))]

    def reseq(a):
        a["seq"] = np.arange(a.size, dtype=np.uint64) + np.uint64(1)
        return a

    def pick(mask):
        idx = np.nonzero(mask)[0]
        return int(idx[rng.integers(0, idx.size)])
    vic = (ev["code"] == 9) & (ev["arg"] != 0)
    if kind == "event_after_victim_demotion":            # demoted is terminal: the claim cannot be offloaded afterwards
        i = pick(vic)
        rec = np.zeros(1, TRACE_DTYPE)
        rec["claim_id"], rec["code"], rec["aux"] = ev["claim_id"][i], 3, 30
        return reseq(np.concatenate([ev[:i + 1], rec, ev[i + 1:]]))
    if kind == "victim_demotion_without_request":        # a resident claim demoted with arg = 0: no request to attribute it to
        ev["arg"][pick(vic)] = 0
    elif kind == "short_run":                            # fewer records than announced
        return reseq(np.delete(ev, run[-1])) if len(run) >= 2 else _set(ev, run, "aux", REQ_FLAG | 2)
    elif kind == "interrupted_conflict_run":
        if len(run) < 2:
            return _set(ev, run, "aux", REQ_FLAG | 2)
        rec = np.zeros(1, TRACE_DTYPE)
        rec["claim_id"], rec["code"] = ev["claim_id"][run[0]], T_USE
        return reseq(np.concatenate([ev[:run[1]], rec, ev[run[1]:]]))
    elif kind == "conflict_names_offloaded_claim":       # only a resident claim can block (resident footprint)
        i = run[0]
        rec = np.zeros(1, TRACE_DTYPE)
        rec["claim_id"], rec["code"], rec["aux"] = ev["claim_id"][i], 3, 30
        return reseq(np.concatenate([ev[:i], rec, ev[i:]]))
    elif kind == "claim_named_twice":
        if len(run) < 2:
            return _set(ev, run, "aux", REQ_FLAG | 2)
        ev["claim_id"][run[-1]] = ev["claim_id"][run[0]]
    elif kind == "extra_conflict_record":                # one record more than announced
        return reseq(np.concatenate([ev[:run[-1] + 1], ev[run[-1]:run[-1] + 1], ev[run[-1] + 1:]]))
    elif kind == "conflict_without_flag":
        ev["aux"][run[0]] = len(run)
    elif kind == "failed_restore_demotion_with_request":  # DEMOTED after RESTORATION_FAILED keeps arg = 0
        i = pick((ev["code"] == 9) & (ev["arg"] == 0))
        ev["arg"][i] = 4242
    else:
        raise ValueError(kind)
    return ev


def _set(ev, run, field, val):
    ev[field][run] = val
    return ev
