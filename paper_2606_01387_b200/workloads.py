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
