"""rc_digest_blocks_noalloc -- the entry point that allocates nothing (include/rc.h) -- against the existing path.

Collected last on purpose (the suite runs with pytest -x): the file name sorts after every other test file.
The no-allocation calls are made first, before any librc context exists in this test, so the entry point is shown to work
without one; the reference values then come from rc_digest_blocks (context, cudaMalloc'd scratch) and, for sampled blocks,
from the oracle.  Bit-exact, like every other parity test here (integer work: no tolerance).  Two calls in a row share the
static scratch: the second is smaller and has a different geometry, so stale partial sums of the first lie all around it."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

from oracle import rco
from paper_2606_01387_b200 import rc


def _outputs(n_blocks, dev):
    return (torch.full((n_blocks,), -1, dtype=torch.int64, device=dev), torch.full((n_blocks,), -1, dtype=torch.int64, device=dev))


def _digests_noalloc(buf, n_blocks, layers, page_bytes, stream, out=None):
    d, e = out if out is not None else _outputs(n_blocks, buf.device)
    code = rc.digest_blocks_noalloc(buf.data_ptr(), n_blocks, layers, page_bytes, d.data_ptr(), e.data_ptr(), stream.cuda_stream)
    return code, d, e


def _digests_context(buf, n_blocks, layers, kv_heads, head_dim, elem_bytes, block_size):
    """The existing path: a context over a dummy one-block pool, rc_digest_blocks on the same bytes."""
    page = block_size * kv_heads * head_dim * elem_bytes
    blk = 2 * layers * page
    pool = torch.zeros(blk, dtype=torch.uint8, device=buf.device)
    fill = torch.zeros(1, dtype=torch.uint8, device=buf.device)
    r = rc.RC(layers, kv_heads, head_dim, elem_bytes, block_size, 1, pool, fill, blk, staging_chunk_bytes=64 * blk,
              max_claims=8, max_table_entries=1 << 12, max_events=64)
    (d, e), _ = r.digest_blocks(buf.data_ptr(), n_blocks, both=True)
    r.close()
    return d, e


def test_no_alloc_digest_matches_the_existing_path_on_two_calls_in_a_row():
    dev = torch.device("cuda:0")
    gen = torch.Generator(device=dev)
    gen.manual_seed(260601387)
    # call 1: Llama-3-8B geometry (32 KiB pages, 64 pages per block), 300 blocks = 19200 pages of the 32768-page scratch
    L1, page1, n1 = 32, 16 * 8 * 128 * 2, 300
    # call 2: Tiny geometry (4 KiB pages: the 4 KiB-tile instantiation), 37 blocks = 148 pages: inside call 1's leftovers
    L2, page2, n2 = 2, 16 * 2 * 64 * 2, 37
    buf1 = torch.randint(0, 256, (n1 * 2 * L1 * page1,), dtype=torch.uint8, device=dev, generator=gen)
    buf2 = torch.randint(0, 256, (n2 * 2 * L2 * page2,), dtype=torch.uint8, device=dev, generator=gen)
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    outs = [_outputs(n1, dev), _outputs(n2, dev), _outputs(n1, dev)]          # the caller owns inputs and outputs
    assert _digests_noalloc(buf2, 1, L2, page2, s)[0] == 0                    # first call on this device: loads the module
    s.synchronize()                                                           # (and with it the 4 MiB static scratch)
    free_before = torch.cuda.mem_get_info()[0]
    c1, d1, e1 = _digests_noalloc(buf1, n1, L1, page1, s, outs[0])
    c2, d2, e2 = _digests_noalloc(buf2, n2, L2, page2, s, outs[1])            # same stream: ordered behind call 1, no overlap
    c3, d3, e3 = _digests_noalloc(buf1, n1, L1, page1, s, outs[2])            # and call 1 once more over call 2's leftovers
    s.synchronize()
    assert (c1, c2, c3) == (0, 0, 0)
    assert free_before - torch.cuda.mem_get_info()[0] < (1 << 20)             # the three calls allocated no device memory
    got = [(x.cpu().numpy().view(np.uint64), y.cpu().numpy().view(np.uint64)) for x, y in ((d1, e1), (d2, e2), (d3, e3))]

    want1 = _digests_context(buf1, n1, L1, 8, 128, 2, 16)
    want2 = _digests_context(buf2, n2, L2, 2, 64, 2, 16)
    for (gd, ge), (wd, we) in ((got[0], want1), (got[1], want2), (got[2], want1)):
        assert np.array_equal(gd, wd) and np.array_equal(ge, we)
    # pinned to the oracle as well, on sampled blocks of both geometries
    h1, h2 = buf1.cpu().numpy(), buf2.cpu().numpy()
    for i in (0, 151, n1 - 1):
        b = h1[i * 2 * L1 * page1:(i + 1) * 2 * L1 * page1]
        assert int(got[0][0][i]) == rco.block_digest(b, 2 * L1, 0) and int(got[0][1][i]) == rco.block_digest(b, 2 * L1, 1)
    for i in (0, 17, n2 - 1):
        b = h2[i * 2 * L2 * page2:(i + 1) * 2 * L2 * page2]
        assert int(got[1][0][i]) == rco.block_digest(b, 2 * L2, 0) and int(got[1][1][i]) == rco.block_digest(b, 2 * L2, 1)


def test_no_alloc_digest_rejects_sizes_beyond_its_scratch_and_bad_arguments():
    dev = torch.device("cuda:0")
    L, page = 2, 4096
    n_max = rc.NOALLOC_MAX_PAGES // (2 * L)
    buf = torch.zeros((n_max + 1) * 2 * L * page, dtype=torch.uint8, device=dev)
    s = torch.cuda.current_stream()
    code, d, e = _digests_noalloc(buf, n_max + 1, L, page, s)
    torch.cuda.synchronize()
    assert code == rc.ERR_TOO_LARGE and "scratch" in rc.lib().rc_strerror(code).decode()
    assert bool((d == -1).all()) and bool((e == -1).all())          # nothing was enqueued
    code, d, e = _digests_noalloc(buf, n_max, L, page, s)           # exactly the maximum is served
    torch.cuda.synchronize()
    assert code == 0 and bool((d != -1).all())
    assert bool((d == d[0]).all()) and bool((e == e[0]).all())      # identical (all-zero) blocks, identical digests
    z = buf.cpu().numpy()[: 2 * L * page]
    assert int(d[0].cpu().numpy().view(np.uint64)) == rco.block_digest(z, 2 * L, 0)
    assert rc.digest_blocks_noalloc(buf.data_ptr(), 1, L, 4096 + 512, d.data_ptr(), e.data_ptr(), 0) == rc.ERR_INVALID
    assert rc.digest_blocks_noalloc(buf.data_ptr() + 8, 1, L, page, d.data_ptr(), e.data_ptr(), 0) == rc.ERR_INVALID
    assert rc.digest_blocks_noalloc(buf.data_ptr(), 1, L, page, 0, e.data_ptr(), 0) == rc.ERR_INVALID
    assert rc.digest_blocks_noalloc(0, 0, L, page, 0, 0, 0) == 0    # empty range: nothing to do
