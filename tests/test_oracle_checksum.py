"""Pins for the oracle's checksum (build-defined: BASELINE.json north_star (d)).

The checksum is not in the paper, so it is pinned by (1) an independent big-int
restatement below that shares nothing with oracle/ (Python ints, explicit masks),
(2) literal golden values in tests/golden/checksum.txt (DESIGN.md "Checksum",
SURVEY §8(c).3), (3) closed forms and invariants.
"""
import os

import numpy as np
import pytest

from oracle import rco

M64 = (1 << 64) - 1
C1, C2, A, C3 = 0x9E3779B97F4A7C15, 0x6A09E667F3BCC909, 0xBB67AE8584CAA73B, 0x3C6EF372FE94F82B


def mixL(x):
    y = x ^ (x >> 32)
    y = (y * C2) & M64
    return y ^ (y >> 29)


def mixF(x):
    y = (mixL(x) * C1) & M64
    return y ^ (y >> 32)


def page_digest_py(b: bytes):
    V = len(b) // 16
    w = [int.from_bytes(b[8 * i:8 * i + 8], "little") for i in range(2 * V)]
    p = 0
    for lane in range(256):
        h = ((lane + 1) * C1) & M64
        for v in range(lane, V, 256):
            h = ((h ^ w[2 * v]) * C2) & M64
            h = ((h ^ w[2 * v + 1]) * C2) & M64
        p = (p + mixL(h)) & M64
    return p


def block_digest_py(b: bytes, n_pages):
    pg = len(b) // n_pages
    s = 0
    for g in range(n_pages):
        s = (s + mixL(page_digest_py(b[g * pg:(g + 1) * pg]) ^ (((g + 1) * C3) & M64))) & M64
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


def test_golden_values():
    g = golden()
    assert rco.mixL(0) == g["mixL(0)"] == 0
    assert rco.mixL(1) == g["mixL(1)"]
    assert rco.mixF(1) == g["mixF(1)"]
    z = np.zeros(4096, np.uint8)
    assert rco.page_digest(z) == g["page_digest(zero4096)"]
    ramp = (np.arange(4096) & 0xFF).astype(np.uint8)
    assert rco.page_digest(ramp) == g["page_digest(ramp4096)"]
    zb = np.zeros(4 * 4096, np.uint8)
    dz = rco.block_digest(zb, 4)
    assert dz == g["block_digest(tiny zero block)"]
    assert rco.chain_of(1, []) == g["chain_seed(1)"]
    assert rco.chain_of(1, [dz]) == g["chain_of(1,[dz])"]
    assert rco.chain_of(1, [dz, dz]) == g["chain_of(1,[dz,dz])"]


def test_against_bigint_restatement():
    rng = np.random.default_rng(5)
    for x in [0, 1, M64, 0x8000000000000000] + [int(v) for v in rng.integers(0, 1 << 63, 50, dtype=np.uint64)]:
        assert rco.mixL(x) == mixL(x)
        assert rco.mixF(x) == mixF(x)
    for size in (4096, 8192, 16384):
        pg = rng.integers(0, 256, size, dtype=np.uint8)
        assert rco.page_digest(pg) == page_digest_py(pg.tobytes())
    blk = rng.integers(0, 256, 4 * 4096, dtype=np.uint8)
    assert rco.block_digest(blk, 4) == block_digest_py(blk.tobytes(), 4)
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
    base = rco.page_digest(pg)
    seen = set()
    for byte in range(4096):
        for bit in range(8):
            pg[byte] ^= 1 << bit
            dgst = rco.page_digest(pg)
            pg[byte] ^= 1 << bit
            assert dgst != base
            seen.add(dgst)
    # distinct flips may collide with EACH OTHER (top-bit flips of two words of one lane do);
    # the property the design needs is only that none collides with the clean page
    assert len(seen) > 4096 * 7


def test_swaps_are_visible():
    rng = np.random.default_rng(9)
    blk = rng.integers(0, 256, 4 * 4096, dtype=np.uint8)
    base = rco.block_digest(blk, 4)
    v = blk.reshape(-1, 16).copy()
    v[[3, 4]] = v[[4, 3]]                       # two vectors across lanes
    assert rco.block_digest(v.reshape(-1), 4) != base
    v = blk.reshape(-1, 16).copy()
    v[[3, 259]] = v[[259, 3]]                   # two vectors of the same lane (order within lane)
    assert rco.page_digest(v.reshape(-1)[:8192]) != rco.page_digest(blk[:8192])
    p = blk.reshape(4, 4096).copy()
    p[[0, 1]] = p[[1, 0]]                       # two pages
    assert rco.block_digest(p.reshape(-1), 4) != base
    d = [5, 6, 7]
    assert rco.chain_of(1, d) != rco.chain_of(1, [6, 5, 7])   # two blocks
    assert rco.chain_of(1, d) != rco.chain_of(2, d)           # claim id
