"""NEXT-4 GPU parity: TP-sharded restore with a common verdict (DESIGN.md 8 / R24).  Two kv_head shards
are two librc contexts on the one GPU of this box, called one after the other from one process -- no kernel of one
rank ever waits for the other (rc.h) -- each against an oracle over the same shard.  Checked per rank: local verdict
records, statuses, events (byte-identical across ranks and equal to the oracle's), allocator state, fill, pool bytes of
live blocks; through the all-gather form of the commit and through the peer-mailbox form (k_tp_push stores into the
other context's mailbox; the commit refuses with RC_ERR_BUSY until every rank has published)."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

from oracle import rco, validator as V
from paper_2606_01387_b200 import rc, tp

import tp_inputs as T

XFER, FLIP = 1, 2


class Rank:
    def __init__(self, full, tabs, fill, rank):
        self.part_h = T.shard(full, rank).copy()
        self.pool_t = torch.from_numpy(self.part_h.copy()).cuda()
        self.fill_h = np.zeros(T.NB, np.uint8)
        self.fill_t = torch.zeros(T.NB, dtype=torch.uint8, device="cuda")
        self.fill_t[:] = torch.from_numpy(fill).cuda()
        torch.cuda.synchronize()
        hs = T.H // T.G
        self.o = rco.Oracle(T.L, hs, T.D, T.E, T.BS, T.NB, self.part_h, self.fill_h)
        self.o.set_tp(T.G)
        blk = 2 * T.L * T.BS * hs * T.D * T.E
        self.r = rc.RC(T.L, hs, T.D, T.E, T.BS, T.NB, self.pool_t, self.fill_t, 1 << 28, staging_chunk_bytes=7 * blk,
                       tp_ranks=T.G, tp_rank=rank)
        self.ids = T.admit(self.o, tabs, self.fill_h, fill)
        assert T.admit(self.r, tabs, np.zeros(T.NB, np.uint8), fill) == self.ids
        assert np.array_equal(self.o.offload(self.ids), self.r.offload(self.ids))
        self.blk = blk

    def poison(self):
        used, _ = self.o.pool_state()
        free = np.nonzero(used == 0)[0]
        hv = self.part_h.reshape(2 * T.L, T.NB, -1)
        hv[:, free, :] = 0xA5
        self.pool_t.view(2 * T.L, T.NB, -1)[:, torch.from_numpy(free.astype(np.int64)).cuda(), :] = 0xA5
        torch.cuda.synchronize()

    def check(self, what):
        for c in self.ids:
            assert self.o.claim_info(c) == self.r.claim_info(c), (what, hex(c))
            assert np.array_equal(self.o.claim_blocks(c), self.r.claim_blocks(c)), what
        ua, ra = self.o.pool_state()
        ub, rb = self.r.pool_state()
        assert np.array_equal(ua, ub) and np.array_equal(ra, rb), what
        assert np.array_equal(self.fill_h, self.fill_t.cpu().numpy()), what
        live = np.nonzero(ua == 1)[0]
        got = self.pool_t.view(2 * T.L, T.NB, -1)[:, torch.from_numpy(live.astype(np.int64)).cuda(), :].cpu().numpy()
        assert np.array_equal(got, self.part_h.reshape(2 * T.L, T.NB, -1)[:, live, :]), what


def faults_of(ranks, ids):
    b = ranks[0].blk
    return [[(ids[2], FLIP, 5 * b + 17), (ids[3], XFER, 0)], [(ids[1], XFER, 0), (ids[2], FLIP, 2 * b + 99), (ids[3], FLIP, 4 * b)]]


def test_tp_restore_all_gather_form():
    full, tabs, fill = T.make()
    ranks = [Rank(full, tabs, fill, r) for r in range(T.G)]
    ids = ranks[0].ids
    loc_o, loc_r, st_o, st_r = [], [], [], []
    for rk, f in zip(ranks, faults_of(ranks, ids)):
        rk.poison()
        assert rk.o.set_faults(f) == 0 and rk.r.set_faults(f) == 0
        so, vo = rk.o.tp_restore_verify(ids)
        sr, vr = rk.r.tp_restore_verify(ids)
        assert np.array_equal(so, sr) and np.array_equal(vo, vr), (vo, vr)      # local verdicts, record by record
        assert len(rk.r.outcomes()) == len(rk.o.outcomes())                     # drains offload-time events; verify emits none
        rcode, _ = rk.r.restore(ids, check=False)
        assert rcode == rc.ERR_BUSY                                             # the split restore is waiting for its commit
        loc_o.append(vo); loc_r.append(vr); st_o.append(so); st_r.append(sr)
    gathered = np.stack(loc_r)
    bad = gathered.copy()
    bad["flags"][1][0] = 0
    rcode, _ = ranks[0].r.tp_restore_commit(bad, st_r[0].copy(), check=False)
    assert rcode == rc.ERR_INVALID                                              # ranks disagree on `served`: nothing applied
    streams = []
    for rk, so, sr in zip(ranks, st_o, st_r):
        rk.o.tp_restore_commit(np.stack(loc_o), so)
        rk.r.tp_restore_commit(gathered, sr)
        assert np.array_equal(so, sr) and list(sr) == [0, 8, 8, 8, 0]
        ea, eb = rk.o.outcomes(), rk.r.outcomes()
        assert ea.tobytes() == eb.tobytes()
        streams.append(eb)
        rk.check("commit")
    assert streams[0].tobytes() == streams[1].tobytes()                          # identical emission on every rank
    assert {int(e["claim_id"]): int(e["aux"]) for e in streams[0] if int(e["code"]) == 5} == {
        ids[1]: 0xFFFFFFFF, ids[2]: 2, ids[3]: 4}
    # the shards of the restored claims reassemble to the original full-layout bytes
    parts = [rk.pool_t.cpu().numpy() for rk in ranks]
    re = T.unshard(parts).reshape(T.L * 2, T.NB, -1)
    orig = T.make()[0].reshape(T.L * 2, T.NB, -1)
    for k in (0, 4):
        new = ranks[0].r.claim_blocks(ids[k])
        assert np.array_equal(re[:, new, :], orig[:, tabs[k][: len(new)], :])
    for rk in ranks:
        rk.r.close()


def test_tp_restore_peer_mailbox_form():
    full, tabs, fill = T.make()
    ranks = [Rank(full, tabs, fill, r) for r in range(T.G)]
    ids = ranks[0].ids
    mb = [rk.r.tp_mailbox()[0] for rk in ranks]
    assert ranks[0].r.tp_set_peer(1, mb[1]) == 0 and ranks[1].r.tp_set_peer(0, mb[0]) == 0
    assert ranks[0].r.tp_set_peer(0, mb[0]) != 0                                # own rank / out of range are rejected
    for round_ in range(2):                                                      # two epochs through the same mailboxes
        sel = ids if round_ == 0 else [ids[0], ids[4]]
        if round_ == 1:
            for rk in ranks:
                assert np.array_equal(rk.o.offload(sel), rk.r.offload(sel))
                rk.o.outcomes(); rk.r.outcomes()
        fl = faults_of(ranks, ids) if round_ == 0 else [[], [(ids[4], FLIP, 3)]]
        st_o, st_r, loc_o = [], [], []
        for i, (rk, f) in enumerate(zip(ranks, fl)):
            rk.poison()
            assert rk.o.set_faults(f) == 0 and rk.r.set_faults(f) == 0
            so, vo = rk.o.tp_restore_verify(sel)
            sr, vr = rk.r.tp_restore_verify(sel)                                # pushes into both mailboxes
            assert np.array_equal(vo, vr)
            st_o.append(so); st_r.append(sr); loc_o.append(vo)
            if i == 0:                                                          # rank 1 has not published this epoch yet
                rcode, _ = rk.r.tp_restore_commit(None, sr, check=False)
                assert rcode == rc.ERR_BUSY
        for rk, so, sr in zip(ranks, st_o, st_r):
            rk.o.tp_restore_commit(np.stack(loc_o), so)
            rk.r.tp_restore_commit(None, sr)                                    # merged from this rank's own mailbox
            assert np.array_equal(so, sr)
            assert rk.o.outcomes().tobytes() == rk.r.outcomes().tobytes()
            rk.check("mailbox commit %d" % round_)
        assert list(st_r[0]) == ([0, 8, 8, 8, 0] if round_ == 0 else [0, 8])
    for rk in ranks:
        rk.r.close()


def _ipc_worker(rank, world, port, q):
    import os, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path.insert(0, root); sys.path.insert(0, os.path.join(root, "tests"))
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RC_NO_BUILD="1")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    full, tabs, fill = T.make()
    rk = Rank(full, tabs, fill, rank)
    tp.open_peer_mailboxes(rk.r, dist)                     # CUDA IPC handles over the control plane
    f = faults_of([rk, rk], rk.ids)[rank]
    rk.poison()
    rk.r.set_faults(f)
    st = tp.tp_restore_mailbox(rk.r, rk.ids, dist)         # verify (peer stores) -> barrier -> commit from the mailbox
    ev = rk.r.outcomes()
    out = [None] * world
    dist.all_gather_object(out, (ev.tobytes(), [int(s) for s in st]))
    dist.barrier()
    rk.r.close()
    if rank == 0:
        q.put(out)
    dist.destroy_process_group()


def test_tp_restore_two_processes_cuda_ipc_mailboxes():
    """One process per rank, as deployed: the ranks exchange CUDA IPC handles of their mailboxes, each verify stores its
    records into the peer's memory, a host barrier orders verify before commit (no kernel waits for another process).
    Both processes share this box's one GPU; with one GPU per rank the same stores cross NVLink."""
    import socket
    import torch.multiprocessing as mp
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_ipc_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    out = q.get(timeout=240)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    (ev0, st0), (ev1, st1) = out
    assert st0 == st1 == [0, 8, 8, 8, 0] and ev0 == ev1
    ev = np.frombuffer(ev0, rc.EVENT_DTYPE)
    assert [int(e["code"]) for e in ev if int(e["claim_id"]) == T.SPECS[1][0]][-4:] == [4, 5, 7, 8]
