"""bench.py's pipelined schedule (run_pipeline) against a model of the library's rules (include/rc.h, split forms):
at most two open offloads (one in dedup / direct mode), one restore in flight, a restore only of claims whose offload has
been completed by rc_wait(0), no call on a claim of an operation in flight, a wave admitted only when its claim ids are
not live and its pool region has been left by the wave that used it before.  No GPU."""
import pytest

import bench


class Model:
    def __init__(self, max_open):
        self.max_open, self.open, self.restore = max_open, [], None
        self.state = {}                     # claim id -> "resident" | "offloading" | "offloaded" | "restoring" | "back"
        self.region = {}                    # pool region -> wave key that occupies it with un-offloaded blocks
        self.log, self.max_seen_open, self.overlap = [], 0, 0

    def admit(self, p):
        assert all(c not in self.state for c in p["ids"]), "claim ids still live"
        assert self.region.get(p["region"]) is None, "pool region still holds the previous wave's blocks"
        self.region[p["region"]] = p["key"]
        for c in p["ids"]:
            self.state[c] = "resident"
        self.log.append(("admit", p["key"]))

    def offload_begin(self, ids):
        assert len(self.open) < self.max_open, "RC_ERR_BUSY"
        assert all(self.state[c] == "resident" for c in ids)
        for c in ids:
            self.state[c] = "offloading"
        self.open.append(list(ids))
        self.max_seen_open = max(self.max_seen_open, len(self.open))

    def wait(self, which):
        if which == 0:
            assert self.open
            for c in self.open.pop(0):
                self.state[c] = "offloaded"
                for r, k in list(self.region.items()):
                    if k is not None and c in self.waves[k]:
                        self.region[r] = None
        else:
            assert self.restore is not None
            for c in self.restore:
                self.state[c] = "back"
            self.restore = None

    def set_faults(self, f):
        pass

    def restore_begin(self, ids):
        assert self.restore is None
        assert all(self.state[c] == "offloaded" for c in ids), "restore of a claim whose offload is not complete"
        for c in ids:
            self.state[c] = "restoring"
        self.restore = list(ids)
        self.overlap = max(self.overlap, len(self.open))
        self.log.append(("restore", tuple(ids)))

    def outcomes(self, cap):
        return []

    def release(self, ids):
        for c in ids:
            assert self.state[c] == "back", "release of a claim in flight"
            del self.state[c]


@pytest.mark.parametrize("n_waves,steps,one_open", [(38, 3, False), (33, 3, False), (3, 4, False), (2, 5, False), (1, 4, False),
                                                   (12, 2, True), (4, 1, False), (5, 1, True)])
def test_schedule_respects_the_librarys_rules(n_waves, steps, one_open):
    # waves as bench.py lays them out: consecutive waves of the sequence alternate between two pool regions, also across
    # passes when the number of waves is odd (Job.prep / prep_alt)
    def make(parity):
        return [dict(ids=[10 * w + i for i in range(3)], faults=[], key=w, region=(w + parity) % 2) for w in range(n_waves)]
    prep, alt = make(0), (make(1) if n_waves % 2 else make(0))
    seq = []
    for _ in range(steps):
        seq += prep if len(seq) % 2 == 0 else alt
    m = Model(1 if one_open else 2)
    m.waves = {w: set(10 * w + i for i in range(3)) for w in range(n_waves)}
    n = bench.run_pipeline(m, seq, m.admit, n_waves, one_open, 1000)
    assert n == 0 and not m.state and not m.open and m.restore is None
    assert [x[1] for x in m.log if x[0] == "restore"] == [tuple(p["ids"]) for p in seq]        # every wave, in order
    if n_waves >= 3 and len(seq) >= 4:
        # steady state: offload(j+1) is open when restore(j) begins, and offload(j+2) is queued behind it right after
        assert m.max_seen_open == (1 if one_open else 2)
        assert m.overlap == (0 if one_open else 1)
