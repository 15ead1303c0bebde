"""Tiny geometry with prefix sharing: inputs of the dedup tests (NEXT-2).  Test infrastructure, inputs only."""
import numpy as np

from paper_2606_01387_b200.workloads import GEOMS, N_PRED, SEED0, ClaimSpec, Geometry, Wave, Workload, _ids


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
