"""Pins for the oracle's checksum (build-defined: BASELINE.json north_star (d), R22).

The checksum is not in the paper, so it is pinned by (1) an independent big-int
restatement below that shares nothing with oracle/ (Python ints, explicit masks),
(2) literal golden values in tests/golden/checksum.txt (written by
tests/golden/make_checksum_golden.py from oracle/ only; mixL / mixF / chain seed are
the literals SURVEY 8(c).3 printed), (3) closed forms and invariants, (4) differential
tests: no pair / triple of flipped bits inside one lane cancels (the structural
collision of the round-1 fold h = (h ^ w) * C2, where two bit-63 flips in one lane
left the digest unchanged).
"""
import os

import numpy as np
import pytest

from oracle import rco

M64 = (1 << 64) - 1
C1, C2, A, C3 = 0x9E3779B97F4A7C15, 0x6A09E667F3BCC909, 0xBB67AE8584CAA73B, 0x3C6EF372FE94F82B
C4, C5 = 0xA54FF53A5F1D36F1, 0x510E527FADE682D1


def mixL(x):
    y = x ^ (x >> 32)
    y = (y * C2) & M64
    return y ^ (y >> 29)


def mixF(x):
    y = (mixL(x) * C1) & M64
    return y ^ (y >> 32)


def mum(x, y):
    p = x * y                                              # exact: Python ints
    return (p & M64) ^ (p >> 64)


def page_digest_py(b: bytes, which=0):
    V = len(b) // 16
    w = [int.from_bytes(b[8 * i:8 * i + 8], "little") for i in range(2 * V)]
    p = 0
    for lane in range(256):
        h = ((lane + 1) * (C4 if which else C1)) & M64
        for v in range(lane, V, 256):
            a, bb = w[2 * v], w[2 * v + 1]
            h = mum(bb ^ C5, a ^ h) if which else mum(a ^ C2, bb ^ h)
        p = (p + mixL(h)) & M64
    return p


def block_digest_py(b: bytes, n_pages, which=0):
    pg = len(b) // n_pages
    s = 0
    for g in range(n_pages):
        key = ((g + 1) * (C5 if which else C3)) & M64
        s = (s + mixL(page_digest_py(b[g * pg:(g + 1) * pg], which) ^ key)) & M64
    return mixF(s)


def chain_py(cid, d):
    h = mixF(cid ^ C3)
    for x in d:
        h = (h * A + x) & M64
    return h


def golden():
    out = {}
    path = os.path.join(os.path.dirname(__file__), "golden", "checksum.txt")
    for line in open(path):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            out[k.strip()] = int(v.strip(), 16)
    return out


def test_constants_are_the_stated_irrationals():
    # C1 = floor(2^64/phi); C2, A, C3 = frac(sqrt 2, 3, 5) * 2^64 (C2 and A forced odd): computed with isqrt
    from math import isqrt
    s5 = isqrt(5 << 128)                                   # floor(sqrt(5) * 2^64)
    assert (s5 - (1 << 64)) >> 1 == C1                     # (sqrt5 - 1)/2 = 1/phi
    assert (isqrt(2 << 128) - (1 << 64)) | 1 == C2
    assert isqrt(3 << 128) - (1 << 64) == A and A & 1
    assert s5 - (2 << 64) == C3
    assert isqrt(7 << 128) - (2 << 64) == C4
    assert isqrt(11 << 128) - (3 << 64) == C5


def test_golden_values():
    g = golden()
    assert rco.mixL(0) == g["mixL(0)"] == 0
    assert rco.mixL(1) == g["mixL(1)"]
    assert rco.mixF(1) == g["mixF(1)"]
    # the three literals SURVEY.md 8(c).3 printed for the parts R22 leaves unchanged
    assert g["mixL(1)"] == 0x6A09E664A3F3FA36 and g["mixF(1)"] == 0xE7036A585AD2C436 and g["chain_seed(1)"] == 0x842F98FCDC0ADE24
    assert rco.mum(3, 5) == g["mum(3,5)"] == 15                      # no overflow: plain product
    assert rco.mum(1 << 63, 6) == g["mum(2^63,6)"] == 3              # 3 * 2^64: low half 0, high half 3
    assert rco.mum(C1, C2) == g["mum(C1,C2)"] == mum(C1, C2)
    z = np.zeros(4096, np.uint8)
    ramp = (np.arange(4096) & 0xFF).astype(np.uint8)
    zb = np.zeros(4 * 4096, np.uint8)
    for which, tag in ((0, "d"), (1, "e")):
        assert rco.page_digest(z, which) == g["page_digest(zero4096)." + tag]
        assert rco.page_digest(ramp, which) == g["page_digest(ramp4096)." + tag]
        assert rco.block_digest(zb, 4, which) == g["block_digest(tiny zero block)." + tag]
    dz = rco.block_digest(zb, 4)
    assert rco.chain_of(1, []) == g["chain_seed(1)"]
    assert rco.chain_of(1, [dz]) == g["chain_of(1,[dz])"]
    assert rco.chain_of(1, [dz, dz]) == g["chain_of(1,[dz,dz])"]


def test_against_bigint_restatement():
    rng = np.random.default_rng(5)
    for x in [0, 1, M64, 0x8000000000000000] + [int(v) for v in rng.integers(0, 1 << 63, 50, dtype=np.uint64)]:
        assert rco.mixL(x) == mixL(x)
        assert rco.mixF(x) == mixF(x)
    for x, y in [(0, 5), (M64, M64), (1 << 63, 1 << 63), (C1, 1)] + [
            (int(a), int(b)) for a, b in rng.integers(0, 1 << 63, (20, 2), dtype=np.uint64) * 2 + 1]:
        assert rco.mum(x, y) == mum(x, y) == mum(y, x)
    for which in (0, 1):
        for size in (4096, 8192, 16384):
            pg = rng.integers(0, 256, size, dtype=np.uint8)
            assert rco.page_digest(pg, which) == page_digest_py(pg.tobytes(), which)
        blk = rng.integers(0, 256, 4 * 4096, dtype=np.uint8)
        assert rco.block_digest(blk, 4, which) == block_digest_py(blk.tobytes(), 4, which)
    d = [int(v) for v in rng.integers(0, 1 << 63, 9, dtype=np.uint64)]
    assert rco.chain_of(0xDEADBEEF, d) == chain_py(0xDEADBEEF, d)


def test_mixers_are_bijections_on_a_sample():
    # x -> x ^ (x >> k) and odd multiplication are invertible; invert explicitly
    def unshift(y, k):
        x = y
        for _ in range(64 // k + 1):
            x = y ^ (x >> k)
        return x
    inv2, inv1 = pow(C2, -1, 1 << 64), pow(C1, -1, 1 << 64)
    for x in [0, 1, 2, M64, 0x0123456789ABCDEF]:
        y = rco.mixL(x)
        assert unshift((unshift(y, 29) * inv2) & M64, 32) == x
        z = rco.mixF(x)
        assert unshift((unshift((unshift(z, 32) * inv1) & M64, 29) * inv2) & M64, 32) == x


def test_chain_closed_form():
    # H_k = seed*A^(k+1) + sum_i d_i * A^(k-i)
    rng = np.random.default_rng(6)
    d = [int(v) for v in rng.integers(0, 1 << 63, 40, dtype=np.uint64)]
    cid = 0x1234
    seed = rco.chain_of(cid, [])
    for k in (0, 1, 7, 39):
        want = (seed * pow(A, k + 1, 1 << 64) + sum(d[i] * pow(A, k - i, 1 << 64) for i in range(k + 1))) & M64
        assert rco.chain_of(cid, d[:k + 1]) == want


def test_chain_scan_combine_is_associative():
    # (a1,b1)*(a2,b2) = (a1*a2, b1*a2 + b2): what a warp scan over (A, d_i) relies on
    rng = np.random.default_rng(7)
    d = [int(v) for v in rng.integers(0, 1 << 63, 33, dtype=np.uint64)]

    def comb(x, y):
        return ((x[0] * y[0]) & M64, (x[1] * y[0] + y[1]) & M64)
    el = [(A, x) for x in d]
    left = el[0]
    for e in el[1:]:
        left = comb(left, e)
    def tree(lo, hi):
        if hi - lo == 1:
            return el[lo]
        mid = (lo + hi) // 2
        return comb(tree(lo, mid), tree(mid, hi))
    assert tree(0, len(el)) == left
    seed = rco.chain_of(99, [])
    assert (seed * left[0] + left[1]) & M64 == rco.chain_of(99, d)


def test_every_single_bit_flip_of_a_page_changes_its_digest():
    rng = np.random.default_rng(8)
    pg = rng.integers(0, 256, 4096, dtype=np.uint8)
    for which in (0, 1):
        base = rco.page_digest(pg, which)
        seen = set()
        for byte in range(4096):
            for bit in range(8):
                pg[byte] ^= 1 << bit
                dgst = rco.page_digest(pg, which)
                pg[byte] ^= 1 << bit
                assert dgst != base
                seen.add(dgst)
        assert len(seen) == 4096 * 8           # and no two single-bit flips collide with each other


def _flip(pg, word, bit):
    pg[8 * word + bit // 8] ^= 1 << (bit % 8)


def test_no_pair_or_triple_of_high_bit_flips_in_one_lane_cancels():
    """The round-1 fold h = (h ^ w) * C2 let a difference in bit 63 travel as exactly 2^63, so a second bit-63 flip in
    any later word of the same lane cancelled it (two bf16 sign bits 8 bytes apart left the digest unchanged).  With the
    mum fold no such structural cancellation exists: every pair of flips among the top bits of the words of one
    lane -- the same vector and the lane's next vector -- changes both digests, and so do the triples that defeat
    a fold with only a downward xor-shift (bit 63 of one word, bits 63 and 31 of the next)."""
    rng = np.random.default_rng(18)
    pg = rng.integers(0, 256, 8192, dtype=np.uint8)     # 512 vectors: lane 5 holds vectors 5 and 261
    base = [rco.page_digest(pg, w) for w in (0, 1)]
    words = [10, 11, 522, 523]                           # the four u64 words of lane 5, in fold order
    tops = (63, 62, 61, 47, 32, 31, 15, 0)
    n = 0
    for i, wa in enumerate(words):
        for wb in words[i:]:
            for ba in tops:
                for bb in tops:
                    if wa == wb and ba >= bb:
                        continue
                    _flip(pg, wa, ba); _flip(pg, wb, bb)
                    for w in (0, 1):
                        assert rco.page_digest(pg, w) != base[w], (wa, ba, wb, bb, w)
                    _flip(pg, wa, ba); _flip(pg, wb, bb)
                    n += 1
    assert n == 496                                       # 6 word pairs x 64 + 4 words x 28 in-word pairs
    for wa, wb in ((10, 11), (11, 522), (522, 523), (10, 522)):
        _flip(pg, wa, 63); _flip(pg, wb, 63); _flip(pg, wb, 31)
        for w in (0, 1):
            assert rco.page_digest(pg, w) != base[w]
        _flip(pg, wa, 63); _flip(pg, wb, 63); _flip(pg, wb, 31)
    # the exact corruption ADVICE r1 reports: MSB of bytes 7 and 15 of one 16-byte vector (two bf16 sign bits)
    pg[16 * 5 + 7] ^= 0x80; pg[16 * 5 + 15] ^= 0x80
    assert rco.page_digest(pg, 0) != base[0] and rco.page_digest(pg, 1) != base[1]


def test_all_pairs_of_bit_flips_inside_one_vector_change_the_digest():
    rng = np.random.default_rng(19)
    pg = rng.integers(0, 256, 4096, dtype=np.uint8)
    base = rco.page_digest(pg, 0)
    v = 77
    seen = set()
    for i in range(128):
        for j in range(i + 1, 128):
            pg[16 * v + i // 8] ^= 1 << (i % 8); pg[16 * v + j // 8] ^= 1 << (j % 8)
            d = rco.page_digest(pg, 0)
            pg[16 * v + i // 8] ^= 1 << (i % 8); pg[16 * v + j // 8] ^= 1 << (j % 8)
            assert d != base
            seen.add(d)
    assert len(seen) == 128 * 127 // 2


def test_the_two_digest_families_are_independent_functions():
    """(d, e) is the 128-bit content key of the dedup store: e must not be a function of d.  Pages that agree in d's
    lane inputs but not in e's cannot be built by hand, so check the weaker, checkable facts: the two differ on every
    sample, swapping the two words of every vector (a <-> b, which maps one family's argument order onto the other's)
    changes both, and a change of one bit moves the two digests by unrelated amounts."""
    rng = np.random.default_rng(20)
    deltas = set()
    for _ in range(40):
        pg = rng.integers(0, 256, 4096, dtype=np.uint8)
        d, e = rco.page_digest(pg, 0), rco.page_digest(pg, 1)
        assert d != e
        sw = pg.reshape(-1, 2, 8)[:, ::-1, :].reshape(-1).copy()
        assert rco.page_digest(sw, 0) not in (d, e) and rco.page_digest(sw, 1) not in (d, e)
        pg[int(rng.integers(0, 4096))] ^= 1 << int(rng.integers(0, 8))
        deltas.add(((rco.page_digest(pg, 0) - d) & M64) ^ ((rco.page_digest(pg, 1) - e) & M64))
    assert len(deltas) == 40


def test_swaps_are_visible():
    rng = np.random.default_rng(9)
    blk = rng.integers(0, 256, 4 * 4096, dtype=np.uint8)
    base = rco.block_digest(blk, 4)
    v = blk.reshape(-1, 16).copy()
    v[[3, 4]] = v[[4, 3]]                       # two vectors across lanes
    assert rco.block_digest(v.reshape(-1), 4) != base
    assert rco.block_digest(v.reshape(-1), 4, 1) != rco.block_digest(blk, 4, 1)
    v = blk.reshape(-1, 16).copy()
    v[[3, 259]] = v[[259, 3]]                   # two vectors of the same lane (order within lane)
    for which in (0, 1):
        assert rco.page_digest(v.reshape(-1)[:8192], which) != rco.page_digest(blk[:8192], which)
    v = blk.reshape(-1, 2, 8).copy()
    v[3] = v[3, ::-1].copy()                    # the two words of one vector
    for which in (0, 1):
        assert rco.page_digest(v.reshape(-1)[:4096], which) != rco.page_digest(blk[:4096], which)
    p = blk.reshape(4, 4096).copy()
    p[[0, 1]] = p[[1, 0]]                       # two pages
    assert rco.block_digest(p.reshape(-1), 4) != base
    assert rco.block_digest(p.reshape(-1), 4, 1) != rco.block_digest(blk, 4, 1)
    d = [5, 6, 7]
    assert rco.chain_of(1, d) != rco.chain_of(1, [6, 5, 7])   # two blocks
    assert rco.chain_of(1, d) != rco.chain_of(2, d)           # claim id
