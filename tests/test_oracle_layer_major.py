"""Pins for the layer-major host layout in the oracle (NEXT-4; reading R28).

Layer-major mode changes where a page sits in a claim's host copy -- [g][block][page] instead of [block][g][page] -- and
nothing else.  Pinned here: the host copy is exactly that permutation of the block-major copy (numpy transpose, not the
oracle's own offset formula); digests, chains, statuses, events, allocation and the restored pool bytes are identical in
both modes; an injected bit flip names the block that the stated layout puts at the flipped byte."""
import numpy as np
import pytest

from conftest import build_tiny_oracle
from oracle import rco
from paper_2606_01387_b200 import workloads as W


def run(layer_major, fault=None):
    o, wl, wave, pool, fill = build_tiny_oracle()
    if layer_major:
        assert o.set_layer_major(True) == 0
    ids = [c.claim_id for c in wl.claims]
    o.accept(ids, [c.P for c in wl.claims], [c.N for c in wl.claims], wave.bt_off, wave.bt_ids)
    st = o.materialize(ids)
    ok = [c for c, s in zip(ids, st) if s == 0]
    assert not o.offload(ok).any()
    host = {c: o.host_read(c).copy() for c in ok}
    dig = {c: o.claim_digests(c, both=True) for c in ok}
    chain = {c: o.claim_info(c)["chain"] for c in ok}
    g = wl.geom
    view = pool.reshape(2 * g.layers, g.pool_blocks, g.page_bytes)
    used, _ = o.pool_state()
    view[:, used == 0, :] = W.POISON
    if fault:
        o.set_faults([(ok[fault[0]], W.FK_BITFLIP, fault[1])])
    st_r = o.restore(ok)
    return o, wl, ok, host, dig, chain, [int(s) for s in st_r], pool


def test_host_copy_is_the_stated_permutation_and_nothing_else_changes():
    a = run(False)
    b = run(True)
    g = a[1].geom
    G, page = 2 * g.layers, g.page_bytes
    for c in a[2]:
        nb = a[0].claim_info(c)["nb"]
        bm = a[3][c].reshape(nb, G, page)                        # block-major: [block][g][page]
        assert np.array_equal(b[3][c], bm.transpose(1, 0, 2).reshape(-1))   # layer-major: [g][block][page]
        assert nb > 1 and not np.array_equal(b[3][c], a[3][c])
        assert np.array_equal(a[4][c][0], b[4][c][0]) and np.array_equal(a[4][c][1], b[4][c][1])   # d and e
        assert a[5][c] == b[5][c]                                  # chain
        assert np.array_equal(a[0].claim_blocks(c), b[0].claim_blocks(c))
    assert a[6] == b[6] and set(a[6]) == {0}
    assert np.array_equal(a[0].outcomes(), b[0].outcomes())
    assert np.array_equal(a[7], b[7])                              # restored pool bytes, freed blocks poisoned
    for x, y in zip(a[0].pool_state(), b[0].pool_state()):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("which", [0, 2])
def test_bit_flip_names_the_block_the_layout_puts_at_that_byte(which):
    o, wl, ok, *_ = run(False)
    g = wl.geom
    G, page, blk = 2 * g.layers, g.page_bytes, g.blk_bytes
    nb = o.claim_info(ok[which])["nb"]
    p = 3 * nb * page + 5 * page + 17                              # layer-major: plane 3, block 5; block-major: block p // blk
    assert p < nb * blk and p // blk != 5
    for lm, want in ((False, p // blk), (True, 5)):
        o, wl, ok, host, dig, chain, st, pool = run(lm, fault=(which, p))
        assert st[which] == 8 and st.count(8) == 1
        ev = o.outcomes()
        bad = [int(e["aux"]) for e in ev if int(e["code"]) == 5]
        assert bad == [want]


def test_mode_switch_is_refused_while_bytes_are_held_and_with_dedup():
    o, wl, wave, pool, fill = build_tiny_oracle()
    assert o.set_dedup(True) == 0 and o.set_layer_major(True) != 0
    assert o.set_dedup(False) == 0 and o.set_layer_major(True) == 0 and o.set_dedup(True) != 0
    ids = [c.claim_id for c in wl.claims]
    o.accept(ids, [c.P for c in wl.claims], [c.N for c in wl.claims], wave.bt_off, wave.bt_ids)
    o.materialize(ids)
    o.offload(ids[:2])
    assert o.set_layer_major(False) != 0
