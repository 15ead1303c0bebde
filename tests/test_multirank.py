"""N>1 path of bench.py on CPU: world_size 2, gloo.  Claims shard by replica with no data-path collective;
the only cross-rank step is the reduction of the timed region (max) and of the units processed (sum)."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.reduce_scalar(dist, 100.0 + 50.0 * rank, "max", device="cpu")
    units = bench.reduce_scalar(dist, 1000.0 * (rank + 1), "sum", device="cpu")
    dist.barrier()
    if rank == 0:
        out.put((ms, units))
    dist.destroy_process_group()


def test_world_size_2_gloo_reduction():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    got = [q.get(timeout=120) for _ in range(1)]
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got[0] == (150.0, 3000.0)                   # max over ranks of the time, sum over ranks of the units
