"""Seeded synthetic workloads for BASELINE.json configs[0..4].

Input generation only: geometry, claim ids, prefix lengths, block tables, `fill`
vectors, fault lists and pool bytes.  None of the method's arithmetic (predicate,
checksum, allocator, event logic) lives here, so the oracle-side tests and the
CUDA-side tests may both import it.
The paper measures on no public suite (two small in-process
prompts); everything here is synthetic and shaped after Llama-3 KV geometry as
BASELINE.json states.
"""
from dataclasses import dataclass, field

import numpy as np

SEED0 = 260601387
N_PRED = 448          # the paper's constant, "leading-prefix-at-least-448"
FK_XFER_ERROR, FK_BITFLIP = 1, 2


@dataclass
class Geometry:
    name: str
    layers: int
    kv_heads: int
    head_dim: int
    elem_bytes: int
    block_size: int
    pool_blocks: int
    dtype: str            # "bf16" | "fp8"

    @property
    def page_bytes(self):
        return self.block_size * self.kv_heads * self.head_dim * self.elem_bytes

    @property
    def blk_bytes(self):
        return 2 * self.layers * self.page_bytes

    @property
    def pool_bytes(self):
        return self.blk_bytes * self.pool_blocks


GEOMS = [
    Geometry("tiny", 2, 2, 64, 2, 16, 256, "bf16"),
    Geometry("llama3-8b", 32, 8, 128, 2, 16, 8192, "bf16"),
    Geometry("llama3-70b", 80, 8, 128, 2, 16, 20000, "bf16"),
    Geometry("fp8-e4m3", 28, 4, 128, 1, 32, 65536, "fp8"),
    Geometry("long-context", 32, 8, 128, 2, 16, 61440, "bf16"),
]


@dataclass
class ClaimSpec:
    claim_id: int
    P: int
    N: int
    M: int                 # intended leading materialized length (fill is built to give exactly this)
    group: int = -1        # prefix group (config 3), -1 = private
    shared: int = 0        # leading table entries taken from the group's list
    fault: tuple = None    # (kind, param) or None


@dataclass
class Workload:
    index: int
    geom: Geometry
    claims: list
    decoys: list = field(default_factory=list)   # fault entries that must change nothing (config 4)
    batch: int = 0                               # config 5: claims per interleaved batch


def _ids(rng, n):
    ids = set()
    while len(ids) < n:
        v = int(rng.integers(1, 1 << 63, dtype=np.uint64)) | (int(rng.integers(0, 2)) << 63)
        if v:
            ids.add(v)
    return sorted(ids, key=lambda x: (x * 0x9E3779B1) & 0xFFFFFFFF)   # fixed shuffle, not sorted by value


def make_workload(index, n_claims=None, pool_blocks=None, scale=1):
    """configs[index]; n_claims / pool_blocks shrink it for parity tests (same recipe, fewer units);
    scale divides the prefix lengths of config 4 (long context) for the same purpose."""
    g0 = GEOMS[index]
    g = Geometry(**{**g0.__dict__, "pool_blocks": pool_blocks or g0.pool_blocks})
    rng = np.random.default_rng(SEED0 + index)
    BS = g.block_size
    if index == 0:
        n = n_claims or 8
        ids = _ids(rng, n)
        claims = [ClaimSpec(ids[k], int(rng.integers(448, 513)), N_PRED, 0) for k in range(n)]
        for c in claims:
            c.M = c.P
        if n > 6:
            claims[6].M = 400                                    # under-materialized: 25 full blocks, then 0
        if n > 3:
            claims[3].fault = (FK_BITFLIP, int(rng.integers(0, 1 << 31)))
        return Workload(0, g, claims)
    if index == 1:
        n = n_claims or 256
        ids = _ids(rng, n)
        claims = [ClaimSpec(ids[k], int(rng.integers(448, 4097)), N_PRED, 0) for k in range(n)]
        for c in claims:
            c.M = c.P
        nf = max(1, round(0.02 * n))
        for j, k in enumerate(rng.choice(n, nf, replace=False)):
            claims[k].fault = (FK_XFER_ERROR, 0) if j % 2 else (FK_BITFLIP, int(rng.integers(0, 1 << 31)))
        return Workload(1, g, claims)
    if index == 2:
        n = n_claims or 1024
        ids = _ids(rng, n)
        w = np.arange(1, 17, dtype=np.float64) ** -1.1
        w /= w.sum()
        claims = []
        for k in range(n):
            P = int(rng.integers(512, 8193))
            grp = int(rng.choice(16, p=w))
            u = float(rng.uniform(0.5, 1.0))
            c = ClaimSpec(ids[k], P, N_PRED, P, grp, int(u * ((P + BS - 1) // BS)))
            if rng.random() < 0.10:                              # under-materialized, private blocks only
                c.M, c.group, c.shared = int(rng.integers(0, 448)), -1, 0
            claims.append(c)
        ok = [k for k, c in enumerate(claims) if c.M >= c.N]
        for j, k in enumerate(rng.choice(ok, max(1, round(0.01 * n)), replace=False)):
            claims[k].fault = (FK_XFER_ERROR, 0) if j % 2 else (FK_BITFLIP, int(rng.integers(0, 1 << 31)))
        return Workload(2, g, claims)
    if index == 3:
        n = n_claims or 4096
        ids = _ids(rng, n + max(2, n // 40))
        spare, ids = ids[n:], ids[:n]
        claims = [ClaimSpec(ids[k], int(rng.integers(448, 1025)), N_PRED, 0) for k in range(n)]
        for c in claims:
            c.M = c.P
        nf = max(1, round(0.05 * n))
        pick = rng.choice(n, 2 * nf, replace=False)
        for j, k in enumerate(pick[:nf]):
            claims[k].fault = (FK_XFER_ERROR, 0) if j % 2 else (FK_BITFLIP, int(rng.integers(0, 1 << 31)))
        decoys = []
        for j, k in enumerate(pick[nf:]):
            kind = (FK_XFER_ERROR, 0) if j % 2 == 0 else (FK_BITFLIP, 7)
            if j % 3 == 0:
                decoys.append((spare[j % len(spare)],) + kind)   # id never accepted
            elif j % 3 == 1:
                decoys.append((0,) + kind)                        # unclaimed (needs the separate flag)
            else:
                claims[k].M = 300                                 # accepted, PRED_FALSE, never restored
                decoys.append((claims[k].claim_id,) + kind)
        return Workload(3, g, claims, decoys)
    if index == 4:
        n = n_claims or 64
        ids = _ids(rng, n)
        claims = []
        for k in range(n):
            P = int(rng.integers(32768 // scale, 131072 // scale + 1))
            u = float(rng.uniform(0.25, 1.0))
            claims.append(ClaimSpec(ids[k], P, N_PRED, max(N_PRED, int(u * P))))
        return Workload(4, g, claims, batch=8)
    raise ValueError(index)


@dataclass
class Wave:
    claim_idx: list        # indices into workload.claims, in batch order
    bt_off: np.ndarray     # u32[n+1]
    bt_ids: np.ndarray     # u32[sum]
    used_ids: np.ndarray   # distinct physical blocks of this wave (for rc_mark_used)
    fill_ids: np.ndarray   # blocks whose fill is written ...
    fill_val: np.ndarray   # ... and the u8 values
    faults: list           # [(claim_id, kind, param)] real faults of this wave
    claim_bytes: int       # sum over claims of nb*blk that a successful offload moves


def n_table(c, BS):
    return (c.P + BS - 1) // BS


def plan_waves(wl, host_store_bytes, pool_blocks=None, max_claims_per_wave=None):
    """Wave rule: the longest run of consecutive claims whose distinct
    physical blocks fit the (empty) pool and whose offloaded bytes fit the host store.  Tables
    come from a fresh seeded permutation of 0..NB-1; prefix groups (config 3) share the leading
    blocks of a per-wave canonical list."""
    g = wl.geom
    NB = pool_blocks or g.pool_blocks
    BS = g.block_size
    rng = np.random.default_rng(SEED0 + 1000 + wl.index)
    waves, k, n = [], 0, len(wl.claims)
    while k < n:
        perm = rng.permutation(NB).astype(np.uint32)
        cursor, host, groups = 0, 0, {}
        idx, offs, ids, fill = [], [0], [], {}
        while k < n and (max_claims_per_wave is None or len(idx) < max_claims_per_wave):
            c = wl.claims[k]
            nt = n_table(c, BS)
            glist = groups.get(c.group, []) if c.group >= 0 else []
            fresh = (max(0, c.shared - len(glist)) + nt - c.shared) if c.group >= 0 else nt
            nb = (c.M + BS - 1) // BS if c.M >= c.N else 0
            if cursor + fresh > NB or host + nb * g.blk_bytes > host_store_bytes:
                break
            if c.group >= 0:
                while len(glist) < c.shared:
                    glist.append(int(perm[cursor])); cursor += 1
                groups[c.group] = glist
                tab = glist[:c.shared] + [int(b) for b in perm[cursor:cursor + nt - c.shared]]
                cursor += nt - c.shared
            else:
                tab = [int(b) for b in perm[cursor:cursor + nt]]
                cursor += nt
            for i, b in enumerate(tab):                          # fill gives exactly M leading tokens
                cap = min(BS, c.P - i * BS)
                f = min(cap, max(0, c.M - i * BS))
                if i < c.shared:
                    f = BS                                       # shared blocks are full blocks
                fill[b] = max(fill.get(b, 0), f) if i < c.shared else f
            idx.append(k); ids.extend(tab); offs.append(len(ids)); host += nb * g.blk_bytes
            k += 1
        if not idx:
            raise ValueError("claim %d does not fit an empty pool / host store" % k)
        fb = np.array(sorted(fill), dtype=np.uint32)
        waves.append(Wave(idx, np.array(offs, np.uint32), np.array(ids, np.uint32),
                          np.unique(np.array(ids, np.uint32)), fb,
                          np.array([fill[int(b)] for b in fb], np.uint8),
                          [(wl.claims[j].claim_id,) + wl.claims[j].fault for j in idx if wl.claims[j].fault],
                          host))
    return waves


def pool_host(geom, seed=None):
    """Pool bytes on the host with numpy (small pools only): bf16 ~ N(0,1) by truncating fp32, or
    uniform random bytes for fp8.  Returns uint8[L*2*NB*page]."""
    rng = np.random.default_rng(SEED0 + 77 if seed is None else seed)
    if geom.dtype == "fp8":
        return rng.integers(0, 256, geom.pool_bytes, dtype=np.uint8)
    x = rng.standard_normal(geom.pool_bytes // 2, dtype=np.float32)
    return (x.view(np.uint32) >> 16).astype(np.uint16).view(np.uint8)


def pool_torch(geom, device, seed=None):
    """Pool bytes generated on `device` with seeded torch, in chunks.  Returns a uint8 tensor."""
    import torch
    gen = torch.Generator(device=device)
    gen.manual_seed(SEED0 + 77 if seed is None else seed)
    out = torch.empty(geom.pool_bytes, dtype=torch.uint8, device=device)
    step = 1 << 28
    for o in range(0, geom.pool_bytes, step):
        m = min(step, geom.pool_bytes - o)
        if geom.dtype == "fp8":
            out[o:o + m] = torch.randint(0, 256, (m,), dtype=torch.uint8, device=device, generator=gen)
        else:
            out[o:o + m].view(torch.bfloat16).copy_(
                torch.randn(m // 2, dtype=torch.float32, device=device, generator=gen))
    return out


POISON = 0xA5   # byte written over freed blocks between offload and restore (DESIGN R5)


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


def make_shared_tiny(n_claims=6, seed=0, pool_blocks=256):
    """Tiny geometry with prefix sharing (NEXT-2 inputs): claims share their leading blocks physically in
    two groups, and `copies` lists (src, dst) block pairs whose bytes the harness makes identical, so that
    different physical blocks carry the same content.  Returns (Workload, Wave, copies)."""
    g0 = GEOMS[0]
    g = Geometry(**{**g0.__dict__, "pool_blocks": pool_blocks})
    rng = np.random.default_rng(SEED0 + 7000 + seed)
    ids = _ids(rng, n_claims)
    perm = [int(b) for b in rng.permutation(pool_blocks)]
    cur = 0
    groups = {}
    for gi in range(2):
        groups[gi] = perm[cur:cur + 24]
        cur += 24
    claims, offs, tab_all, fill = [], [0], [], {}
    for k in range(n_claims):
        P = int(rng.integers(448, 513))
        nt = (P + g.block_size - 1) // g.block_size
        shared = int(rng.integers(8, 25))
        c = ClaimSpec(ids[k], P, N_PRED, P, k % 2, shared)
        tab = groups[k % 2][:shared] + perm[cur:cur + nt - shared]
        cur += nt - shared
        for i, b in enumerate(tab):
            fill[b] = max(fill.get(b, 0), g.block_size if i < shared else min(g.block_size, P - i * g.block_size))
        claims.append(c)
        tab_all.extend(tab)
        offs.append(len(tab_all))
    copies = [(tab_all[offs[0] + 26], tab_all[offs[1] + 27]), (tab_all[offs[2] + 25], tab_all[offs[2] + 26])]
    fb = np.array(sorted(fill), dtype=np.uint32)
    wave = Wave(list(range(n_claims)), np.array(offs, np.uint32), np.array(tab_all, np.uint32),
                np.unique(np.array(tab_all, np.uint32)), fb, np.array([fill[int(b)] for b in fb], np.uint8), [], 0)
    return Workload(0, g, claims), wave, copies


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
