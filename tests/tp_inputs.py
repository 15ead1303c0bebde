"""Inputs of the TP-sharded tests: a small geometry whose per-rank page is still a multiple of 4096 bytes, claims,
tables and fill.  Inputs only."""
import numpy as np

from paper_2606_01387_b200 import tp

L, H, D, E, BS, NB, G = 2, 4, 64, 2, 16, 96, 2          # full page 8 KiB; H/G = 2 heads per rank: 4 KiB
SPECS = [(0x1111, 200), (0x2222, 160), (0x3333, 230), (0x4444, 100), (0x5555, 180)]     # (claim id, P tokens)


def make(seed=7):
    rng = np.random.default_rng(seed)
    full = rng.integers(0, 256, L * 2 * NB * BS * H * D * E, dtype=np.uint8)
    perm = [int(b) for b in rng.permutation(NB)]
    tabs, cur = [], 0
    for _, P in SPECS:
        nt = -(-P // BS)
        tabs.append(perm[cur:cur + nt])
        cur += nt
    fill = np.zeros(NB, np.uint8)
    for (_, P), t in zip(SPECS, tabs):
        for i, b in enumerate(t):
            fill[b] = min(BS, P - i * BS)
    return full, tabs, fill


def shard(full, rank):
    return tp.shard_kv_heads(full, L, NB, BS, H, D, E, rank, G)


def unshard(parts):
    """[L][2][NB][BS][H/G][D*e] shards -> the full-layout bytes."""
    v = [np.asarray(p).reshape(L, 2, NB, BS, H // G, D * E) for p in parts]
    return np.concatenate(v, axis=4).reshape(-1)


def admit(o, tabs, fill_arr, fill, which=None):
    """which: indices into SPECS of the claims this context owns (claim sharding); default all."""
    which = list(range(len(SPECS))) if which is None else list(which)
    tabs = [tabs[k] for k in which]
    fill_arr[:] = fill
    used = sorted(b for t in tabs for b in t)
    o.mark_used(used)
    ids = [SPECS[k][0] for k in which]
    off = np.cumsum([0] + [len(t) for t in tabs])
    st = o.accept(ids, [SPECS[k][1] for k in which], [64] * len(ids), off, [b for t in tabs for b in t])
    assert not np.asarray(st).any()
    assert not np.asarray(o.materialize(ids)).any()
    return ids
