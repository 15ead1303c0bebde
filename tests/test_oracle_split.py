"""Pins for the split form of restore in the oracle (rco_restore_begin / rco_restore_end; reading R25).

The split form is the two phases of rco_restore with other calls allowed in between: it has no arithmetic of its own.
Pinned here: back to back it IS rco_restore (statuses, events, tables, pool state, host space, link bytes), with and
without a reuse-request id and in dedup mode; with an offload in between, the restore's allocation is the one taken at
_begin, its records follow the offload's in the stream (P:L27 per-claim order intact), and the host copy is held
until _end."""
import numpy as np
import pytest

from conftest import build_tiny_oracle
from oracle import rco, validator as V
from paper_2606_01387_b200 import workloads as W


def prepared(dedup=False):
    o, wl, wave, pool, fill = build_tiny_oracle()
    if dedup:
        assert o.set_dedup(True) == 0
    ids = [c.claim_id for c in wl.claims]
    assert not o.accept(ids, [c.P for c in wl.claims], [c.N for c in wl.claims], wave.bt_off, wave.bt_ids).any()
    st = o.materialize(ids)
    ok = [c for c, s in zip(ids, st) if s == 0]
    return o, wl, ok, pool


def snapshot(o, ids):
    used, ref = o.pool_state()
    return ([o.claim_info(c) for c in ids], [o.claim_blocks(c).tolist() if o.claim_blocks(c) is not None else None for c in ids],
            used.tobytes(), ref.tobytes(), o.stats(), o.link_bytes())


@pytest.mark.parametrize("dedup", [False, True])
@pytest.mark.parametrize("request_id", [0, 77])
def test_back_to_back_the_split_form_is_restore(dedup, request_id):
    runs = []
    for split in (False, True):
        o, wl, ok, pool = prepared(dedup)
        assert not o.offload(ok).any()
        o.set_faults([(ok[1], W.FK_BITFLIP, 12345), (ok[4], W.FK_XFER_ERROR, 0)])
        if split:
            st0 = o.restore_begin(ok, request_id).copy()
            assert [int(s) for s in st0] == [-1] * len(ok)                  # served: decided by _end
            st = o.restore_end()
        else:
            st = o.restore_request(request_id, ok) if request_id else o.restore(ok)
        runs.append(([int(s) for s in st], o.outcomes().tobytes(), snapshot(o, ok), pool.tobytes()))
        o.close()
    assert runs[0] == runs[1]
    assert runs[0][0].count(8) == 2


def test_calls_between_begin_and_end():
    o, wl, ok, pool = prepared()
    a, b = ok[:3], ok[3:]
    assert not o.offload(a).any()
    used0, _ = o.pool_state()
    free0 = np.nonzero(used0 == 0)[0]
    host_before = o.stats()["host_used"]
    o.set_faults([(a[1], W.FK_BITFLIP, 999)])
    o.restore_begin(a)
    # phase 1 took the lowest free ids of the pool as it stood at _begin, in batch order (R6)
    nb = [o.claim_info(c)["nb"] for c in a]
    got = np.concatenate([o.claim_blocks(c) for c in a])
    assert np.array_equal(got, free0[: sum(nb)])
    assert o.stats()["host_used"] == host_before                            # the host copy is held until _end
    assert all(o.claim_info(c)["state"] == 3 for c in a)                    # still OFFLOADED: no record yet
    assert not o.offload(b).any()                                           # another call in between
    assert o.release(a[:1]).tolist() == [3] and o.restore(a[:1]).tolist() == [3]   # a claim in flight answers BAD_STATE (rc.h)
    st = o.restore_end()
    assert [int(s) for s in st] == [0, 8, 0]
    ev = o.outcomes()
    ok_v, why = V.validate(ev)
    assert ok_v, why
    codes = [(int(e["claim_id"]), int(e["code"])) for e in ev]
    first_rr = min(i for i, (c, k) in enumerate(codes) if k == 4)
    last_off = max(i for i, (c, k) in enumerate(codes) if k == 3 and c in b)
    assert last_off < first_rr                                              # stream order = order of the calls' effects
    assert V.failure_outcome_gate(ev, a[1])                                 # the seven steps of P:L27 for the failed claim
    assert o.stats()["host_used"] == sum(o.claim_info(c)["nb"] for c in b) * o.blk
    used, ref = o.pool_state()
    bad_blocks = free0[nb[0]: nb[0] + nb[1]]
    assert not used[bad_blocks].any() and not ref[bad_blocks].any()         # the failed claim's blocks are free again
    with pytest.raises(ValueError):
        o.restore_end()                                                     # nothing pending
    o.close()
