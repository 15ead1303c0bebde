"""N>1 paths on CPU: world_size 2, gloo (run here without a GPU).

(1) bench.py's only collective: max over ranks of the timed region, sum over ranks of the units.
(2) TP-sharded restore: each process is one kv_head shard (an oracle over its half of the heads); the
    processes exchange their verdict records with tp.all_gather_verdicts over gloo -- the same plumbing the NCCL run
    uses -- commit the merged verdict, and must emit byte-identical streams, equal to the unsharded oracle's in
    (seq, claim, code, aux).
(3) Claim-sharded replicas: each process restores its own claims; rank 0 joins the streams by (gpu, seq).
"""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
XFER, FLIP = 1, 2


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import bench
    import tp_inputs as T
    from oracle import rco, validator as V
    from paper_2606_01387_b200 import tp
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.reduce_scalar(dist, 100.0 + 50.0 * rank, "max", device="cpu")
    units = bench.reduce_scalar(dist, 1000.0 * (rank + 1), "sum", device="cpu")

    # ---- (2) TP: this rank's kv_head shard
    full, tabs, fill = T.make()
    part = T.shard(full, rank).copy()
    f = np.zeros(T.NB, np.uint8)
    o = rco.Oracle(T.L, T.H // T.G, T.D, T.E, T.BS, T.NB, part, f)
    o.set_tp(world)
    ids = T.admit(o, tabs, f, fill)
    assert not o.offload(ids).any()
    blk = o.blk
    faults = [[(ids[2], FLIP, 5 * blk + 17), (ids[3], XFER, 0)],
              [(ids[1], XFER, 0), (ids[2], FLIP, 2 * blk + 99), (ids[3], FLIP, 4 * blk)]][rank]
    o.set_faults(faults)
    st = tp.tp_restore(o, ids, dist, "cpu")                    # verify -> all-gather over gloo -> commit
    ev = o.outcomes()
    streams = [None] * world
    dist.all_gather_object(streams, (ev.tobytes(), [int(s) for s in st], o.pool_state()[0].tobytes()))

    # ---- (3) claim sharding: rank r owns claims r, r+world, ... of one workload on its own full pool
    whole = rco.Oracle(T.L, T.H, T.D, T.E, T.BS, T.NB, full.copy(), np.zeros(T.NB, np.uint8))
    mine = T.admit(whole, tabs, whole.fill, fill, which=range(rank, len(ids), world))
    assert mine == ids[rank::world]
    whole.offload(mine)
    whole.set_faults([(mine[0], XFER, 0)])
    whole.restore(mine)
    own = whole.outcomes()
    shards = [None] * world
    dist.all_gather_object(shards, own.tobytes())
    dist.barrier()
    if rank == 0:
        out.put(dict(ms=ms, units=units, streams=streams, shards=shards, ids=ids))
    dist.destroy_process_group()


def test_world_size_2_gloo():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    got = q.get(timeout=300)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert (got["ms"], got["units"]) == (150.0, 3000.0)     # max over ranks of the time, sum over ranks of the units

    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import tp_inputs as T
    from oracle import rco, validator as V
    from paper_2606_01387_b200 import tp
    ids = got["ids"]
    (ev0, st0, used0), (ev1, st1, used1) = got["streams"]
    assert ev0 == ev1 and st0 == st1 == [0, 8, 8, 8, 0] and used0 == used1      # identical emission, verdict, allocation
    ev = np.frombuffer(ev0, rco.EVENT_DTYPE)
    assert V.validate(ev)[0]
    full, tabs, fill = T.make()
    whole = rco.Oracle(T.L, T.H, T.D, T.E, T.BS, T.NB, full, np.zeros(T.NB, np.uint8))
    T.admit(whole, tabs, whole.fill, fill)
    whole.offload(ids)
    whole.set_faults([(ids[1], XFER, 0), (ids[2], FLIP, 2 * whole.blk + 5), (ids[3], FLIP, 4 * whole.blk)])
    whole.restore(ids)
    ew = whole.outcomes()
    for f in ("seq", "claim_id", "code", "aux"):             # equal to the unsharded oracle's stream (chains are rank-local)
        assert np.array_equal(ew[f], ev[f]), f

    per_gpu = [np.frombuffer(b, rco.EVENT_DTYPE) for b in got["shards"]]
    merged, origin = tp.merge_outcomes(per_gpu)
    assert V.validate(merged)[0] and merged.size == sum(s.size for s in per_gpu)
    for g, stream in enumerate(per_gpu):
        for cid in np.unique(stream["claim_id"]):
            assert V.failure_outcome_gate(merged, int(cid)) == V.failure_outcome_gate(stream, int(cid))
    failed = sorted(int(e["claim_id"]) for e in merged if int(e["code"]) == 8)
    assert failed == sorted([ids[0], ids[1]])                # each replica's own injected failure, nobody else's
