"""bench.py -- claim-scoped KV offload+restore throughput on B200 (BASELINE.json metric).

A step is one pass of the whole hot path (accept, materialize, offload, restore, outcomes,
release: SURVEY.md 8(a) rows a0-a8) over every wave of the workload.  Default workload:
BASELINE.json configs[1] (Llama-3-8B KV shape, pool 8192 blocks = 16 GiB, 256 claims of 448-4096
tokens, 2% injected restore failures), synthetic and seeded.  Prints ONE JSON line.

  python bench.py --gpus 1 --steps 3 --warmup 3
  python -m torch.distributed.run --nproc-per-node N ... bench.py --gpus N ...   (claims are independent:
        every rank runs the workload on its own GPU, pool and host link; no data-path collective)
  python bench.py --impl reference      (the oracle, as it stands, on the host cores; bounded sample)
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_01387_b200 import workloads as W  # noqa: E402

METRIC = "kv_offload_restore_throughput"
UNIT = "GB/s"


def peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.th.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i] == "Active"})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def host_ram_bytes():
    try:
        return os.sysconf("SC_PAGE_SIZE") * os.sysconf("SC_PHYS_PAGES")
    except Exception:
        return 64 << 30


def run_pipeline(r, seq, admit, n_distinct, one_open, ev_cap):
    """The pipelined schedule over a sequence of pre-marshalled waves (dicts with "ids" and "faults"); `admit(p)` makes wave
    p resident (fill, mark_used, accept, materialize).  While wave j is restored, waves j+1 and j+2 are offloaded back to
    back (two open offloads, rc.h).  Between the end of restore(j-1) and the first H2D copy of restore(j) stand only:
    rc_wait(0) -- offload(j) takes effect: reference drop, OFFLOADED --, the release of wave j-1 and rc_restore_begin (plan).
    Everything else -- draining the records, admitting wave j+2 (its pool region is the one offload(j) has just left) and
    queueing offload(j+2) behind offload(j+1) -- runs while both directions move data: the metadata stream is idle until
    rc_wait(1) enqueues the restore's verdicts.  Returns the number of records drained.
    `ahead` = how many waves may be admitted beyond the one being restored: wave j+2 of a two-wave workload (j+1 of a
    one-wave workload) carries the claim ids of wave j and can only be admitted after its release; dedup / direct_offload
    allow one open offload."""
    ahead = min(1 if one_open else 2, n_distinct - 1)
    adm = n_ev = 0

    def push():
        nonlocal adm
        admit(seq[adm])
        r.offload_begin(seq[adm]["ids"])
        adm += 1
    for _ in range(min(len(seq), max(1, ahead))):
        push()
    for j, p in enumerate(seq):
        r.wait(0)
        if j > 0 and ahead >= 1:
            r.release(seq[j - 1]["ids"])
        r.set_faults(p["faults"])
        r.restore_begin(p["ids"])
        if j > 0 and ahead >= 1:
            n_ev += len(r.outcomes(cap=ev_cap))
        if ahead >= 1 and adm < len(seq):
            push()
        r.wait(1)
        if ahead == 0:
            n_ev += len(r.outcomes(cap=ev_cap))
            r.release(p["ids"])
            if adm < len(seq):
                push()
    if ahead >= 1 and seq:
        n_ev += len(r.outcomes(cap=ev_cap))
        r.release(seq[-1]["ids"])
    return n_ev


class Job:
    """One rank's workload: context, resident pool, pre-marshalled waves."""

    def __init__(self, index, rank, n_gpus, chunk_bytes, mover, grid_ctas, host_cap=None, pipelined=True, wave_frac=8, dedup=False, direct=False,
                 layer_major=False):
        import torch
        from paper_2606_01387_b200 import rc
        self.torch, self.rc = torch, rc
        self.wl = W.make_workload(index)
        g = self.g = self.wl.geom
        dev = torch.device("cuda", torch.cuda.current_device())
        budget = int(0.5 * host_ram_bytes() / max(1, n_gpus))
        self.host_store = min(g.pool_bytes, budget, host_cap or (64 << 30)) // g.blk_bytes * g.blk_bytes
        # pipelined: restore of wave k overlaps the offload of wave k+1 (full-duplex host link); waves of 1/wave_frac
        # of the pool (>= 2 so that two waves fit) keep the un-overlapped first offload and last restore short;
        # serial: one wave owns the pool and the host store
        self.pipelined = pipelined
        self.one_open = bool(dedup or direct)
        mc = self.wl.batch or None                    # configs[4]: interleaved batches of 8 claims
        if pipelined:
            while True:                               # largest claims (configs[4]: up to 8192 blocks) may need bigger waves
                try:
                    # three waves hold host bytes at a time: restore(j), offload(j+1), offload(j+2)
                    self.waves = W.plan_waves(self.wl, self.host_store // max(4, wave_frac), pool_blocks=g.pool_blocks // wave_frac,
                                              max_claims_per_wave=mc)
                    break
                except ValueError:
                    if wave_frac <= 2:
                        raise
                    wave_frac //= 2
        else:
            self.waves = W.plan_waves(self.wl, self.host_store, max_claims_per_wave=mc)
        self.pool = W.pool_torch(g, dev, seed=W.SEED0 + 77 + rank)
        self.fill = torch.zeros(g.pool_blocks, dtype=torch.uint8, device=dev)
        n_max = max(len(w.claim_idx) for w in self.waves)
        self.r = rc.RC(g.layers, g.kv_heads, g.head_dim, g.elem_bytes, g.block_size, g.pool_blocks, self.pool, self.fill,
                       self.host_store, staging_chunk_bytes=min(chunk_bytes, self.host_store), staging_chunks=2,
                       max_claims=max(1024, 4 * n_max), max_table_entries=max(4 * g.pool_blocks, 1 << 16),
                       max_events=max(1 << 16, 16 * n_max), mover=mover, grid_ctas=grid_ctas, dedup=dedup, direct_offload=direct, layer_major=layer_major)
        region = g.pool_blocks // wave_frac if pipelined else 0
        dev_ = dev

        def marshal(parity):
            out = []
            for wi, w in enumerate(self.waves):
                bt_ids, used_ids, fill_ids = w.bt_ids, w.used_ids, w.fill_ids
                if pipelined:
                    # consecutive waves of the sequence alternate between the two top regions of the pool; restored blocks
                    # (lowest free ids) land below them, so every wave reads pristine, pairwise distinct content (matters
                    # for --dedup: copies left behind by earlier restores must not masquerade as shared prefixes)
                    base = np.uint32(g.pool_blocks - (1 + (wi + parity) % 2) * region)
                    bt_ids, used_ids, fill_ids = bt_ids + base, used_ids + base, fill_ids + base
                cl = [self.wl.claims[k] for k in w.claim_idx]
                ids = np.array([c.claim_id for c in cl], np.uint64)
                fid_h = torch.from_numpy(fill_ids.astype(np.int64)).pin_memory()
                fval_h = torch.from_numpy(w.fill_val.copy()).pin_memory()
                out.append(dict(ids=ids, P=np.array([c.P for c in cl], np.uint32), N=np.array([c.N for c in cl], np.uint32),
                                bt_off=w.bt_off, bt_ids=bt_ids, used=used_ids, faults=w.faults,
                                fid_h=fid_h, fval_h=fval_h, fid_d=fid_h.to(dev_), fval_d=fval_h.to(dev_), n=len(cl),
                                fill_ids=fill_ids.astype(np.uint32), fill_val=w.fill_val.astype(np.uint8)))
            return out
        self.prep = marshal(0)
        # an odd number of waves: every second pass over the workload runs with the regions swapped, so that consecutive
        # waves of the sequence never share a region
        self.prep_alt = marshal(1) if pipelined and len(self.waves) % 2 else self.prep
        self.meta_h2d = sum(p["ids"].nbytes + p["P"].nbytes + p["N"].nbytes + p["bt_off"].nbytes + p["bt_ids"].nbytes +
                            p["used"].nbytes + 4 * p["ids"].nbytes for p in self.prep)   # ids re-sent by 4 more calls
        self.fill_h2d = sum(p["fill_ids"].nbytes + p["fill_val"].nbytes for p in self.prep)
        self.events = 0

    def close(self):
        import gc
        self.r.close()
        self.pool = self.fill = None
        for p in self.prep:
            p.clear()
        gc.collect()
        self.torch.cuda.empty_cache()

    def _admit(self, p, e2e):
        if e2e:     # fill[] arrives as host arrays inside the timed region (rc_set_fill: staged in the library's pinned
            self.r.set_fill(p["fill_ids"], p["fill_val"])     # buffer, moved over PCIe without a copy engine)
        else:       # resident inputs: fill values already in HBM
            self.fill.index_copy_(0, p["fid_d"], p["fval_d"])
            self.torch.cuda.current_stream().synchronize()
        self.r.mark_used(p["used"])
        self.r.accept(p["ids"], p["P"], p["N"], p["bt_off"], p["bt_ids"])
        self.r.materialize(p["ids"])

    def run(self, n_steps, e2e):
        """n_steps passes over the workload's waves.  Pipelined schedule: the waves of all passes form one sequence;
        while wave j is restored, waves j+1 and j+2 are offloaded back to back (two open offloads, rc.h), across pass
        boundaries too.  Metadata steps run in call order, so every observable equals the synchronous calls."""
        r = self.r
        n_ev = 0
        if not self.pipelined:
            for _ in range(n_steps):
                for p in self.prep:
                    self._admit(p, e2e)
                    r.offload(p["ids"])
                    r.set_faults(p["faults"])
                    r.restore(p["ids"])
                    n_ev += len(r.outcomes(cap=8 * p["n"]))
                    r.release(p["ids"])
        else:
            seq = []
            for _ in range(n_steps):
                seq += self.prep if len(seq) % 2 == 0 else self.prep_alt
            nmax = max(p["n"] for p in self.prep)
            n_ev = run_pipeline(r, seq, lambda p: self._admit(p, e2e), len(self.prep), self.one_open, 32 * nmax)
        self.events = n_ev // max(1, n_steps)
        return n_ev

    def step(self, e2e):
        return self.run(1, e2e)


def time_steps(job, steps, warmup, e2e, dist):
    torch = job.torch
    job.run(warmup, e2e)
    job.r.stats_reset()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    e0.record()
    job.run(steps, e2e)
    e1.record()
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    if dist is not None:
        dist.barrier()
    ms = max(e0.elapsed_time(e1), 0.0)
    st = job.r.stats()
    # every claim whose predicate holds went through offload and restore in every step; nothing was skipped for lack of
    # host space or free blocks (statuses are not inspected inside the timed region)
    want = sum(1 for w in job.waves for k in w.claim_idx if job.wl.claims[k].M >= job.wl.claims[k].N) * steps
    if st["claims_offloaded"] != want or st["claims_restored"] + st["claims_refused"] != want:
        raise SystemExit("bench.py: %d claims expected per direction, %d offloaded, %d restored or refused" % (
            want, st["claims_offloaded"], st["claims_restored"] + st["claims_refused"]))
    return ms, wall * 1e3, st


class OracleJob:
    """The oracle (oracle/, plain single-threaded C++) on a bounded sample of the same workload:
    the first `n_claims` claims of the config on a reduced pool, same recipe, same calls.
    shard = (p, P): this process takes claims p, p+P, ... of a P times larger sample (claims are independent)."""

    def __init__(self, index, n_claims, pool_blocks, shard=None):
        from oracle import rco
        if shard is None:
            self.wl = W.make_workload(index, n_claims=n_claims, pool_blocks=pool_blocks)
        else:
            self.wl = W.make_workload(index, n_claims=n_claims * shard[1], pool_blocks=pool_blocks)
            self.wl.claims = self.wl.claims[shard[0]::shard[1]]
            for c in self.wl.claims:                       # prefix groups do not survive sharding: private blocks
                c.group, c.shared = -1, 0
        g = self.g = self.wl.geom
        self.pool = W.pool_host(g)
        self.fill = np.zeros(g.pool_blocks, np.uint8)
        self.host_store = g.pool_bytes
        self.waves = W.plan_waves(self.wl, self.host_store)
        self.o = rco.Oracle(g.layers, g.kv_heads, g.head_dim, g.elem_bytes, g.block_size, g.pool_blocks, self.pool,
                            self.fill, self.host_store)
        self.sample = "first %d claims of configs[%d] on a %d-block pool (%d waves), offload+restore+outcomes" % (
            n_claims, index, pool_blocks, len(self.waves))

    def step(self):
        o, wl = self.o, self.wl
        moved = 0
        for w in self.waves:
            cl = [wl.claims[k] for k in w.claim_idx]
            ids = [c.claim_id for c in cl]
            self.fill[w.fill_ids] = w.fill_val
            o.mark_used(w.used_ids)
            o.accept(ids, [c.P for c in cl], [c.N for c in cl], w.bt_off, w.bt_ids)
            o.materialize(ids)
            st = o.offload(ids)
            nb = sum(o.claim_info(c)["nb"] for c, s in zip(ids, st) if s == 0)
            o.set_faults(w.faults)
            st = o.restore(ids)
            o.outcomes(cap=8 * len(ids))
            moved += nb * self.g.blk_bytes * 2        # once per direction, as the GPU arm counts payload
            o.release(ids)
        return moved


def oracle_sample_shape(index):
    # sized for roughly 10-20 s of single-thread work per pass
    return {0: (8, 256), 1: (16, 640), 2: (4, 800), 3: (256, 2560), 4: (16, 640)}[index]


def _oracle_shard(args):
    index, p, P = args
    n_claims, pool_blocks = oracle_sample_shape(index)
    job = OracleJob(index, n_claims, pool_blocks, shard=(p, P))
    t0 = time.perf_counter()
    moved = job.step()
    return moved, time.perf_counter() - t0, sum(len(w.claim_idx) for w in job.waves)


def run_oracle_all_cores(index):
    """P = nproc independent oracle processes, claims sharded round-robin; aggregate bytes over the
    slowest process's time.  The oracle itself stays single-threaded."""
    import multiprocessing as mp
    P = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    n_claims, pool_blocks = oracle_sample_shape(index)
    need = P * (W.GEOMS[index].blk_bytes * pool_blocks) * 3                    # pool + host copies per process
    while P > 1 and need > 0.5 * host_ram_bytes():
        P //= 2
        need //= 2
    t0 = time.perf_counter()
    with mp.get_context("spawn").Pool(P) as pool:
        res = pool.map(_oracle_shard, [(index, p, P) for p in range(P)])
    wall = time.perf_counter() - t0
    moved, slowest, claims = sum(r[0] for r in res), max(r[1] for r in res), sum(r[2] for r in res)
    return {"value": moved / slowest / 1e9, "unit": UNIT, "cores": P, "kind": "oracle",
            "sample": "%d processes, each %d claims of configs[%d] (round-robin shard of the first %d) on a %d-block pool" % (
                P, n_claims, index, n_claims * P, pool_blocks),
            "claims_per_s": claims / slowest, "seconds": slowest, "wall_seconds_with_setup": wall}


def run_oracle(index, steps, warmup):
    n_claims, pool_blocks = oracle_sample_shape(index)
    job = OracleJob(index, n_claims, pool_blocks)
    for _ in range(warmup):
        job.step()
    t0 = time.perf_counter()
    moved = 0
    for _ in range(steps):
        moved += job.step()
    dt = time.perf_counter() - t0
    claims = sum(len(w.claim_idx) for w in job.waves) * steps
    return {"value": moved / dt / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": job.sample,
            "claims_per_s": claims / dt, "seconds": dt, "steps": steps}


def single_claim_latency(job, reps=12):
    """Latency of the synchronous calls on ONE claim (the shape of the paper's running example: a reuse request that needs
    an ordered restoration of one claim), wall clock around each call, medians.  Not part of `value`."""
    r, p = job.r, job.prep[0]
    job._admit(p, False)
    k = int(np.argmin(p["P"]))
    cid = p["ids"][k:k + 1]
    r.set_faults([])
    t_off, t_res = [], []
    for _ in range(reps):
        t0 = time.perf_counter(); r.offload(cid); t1 = time.perf_counter(); r.restore(cid); t2 = time.perf_counter()
        t_off.append(t1 - t0); t_res.append(t2 - t1)
        r.outcomes(cap=64)
    info = r.claim_info(int(cid[0]))
    r.release(p["ids"])
    r.outcomes(cap=1 << 16)
    nbytes = info["nb"] * job.g.blk_bytes
    mo, mr = float(np.median(t_off[2:])), float(np.median(t_res[2:]))
    return {"tokens": int(p["P"][k]), "blocks": info["nb"], "bytes": nbytes, "offload_ms": mo * 1e3, "restore_ms": mr * 1e3,
            "offload_gbs": nbytes / mo / 1e9, "restore_gbs": nbytes / mr / 1e9,
            "what": "rc_offload / rc_restore of one claim, synchronous calls, wall clock, median of %d" % (reps - 2)}


def reduce_scalar(dist, x, op, device="cuda"):
    """Cross-rank reduction of one number (the only collective of the multi-GPU run): max for times, sum for units."""
    if dist is None:
        return x
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return float(t.item())


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs index (1 = the metric's workload)")
    ap.add_argument("--chunk-mib", type=int, default=2048)
    ap.add_argument("--mover", default="auto", choices=["auto", "ldg", "tma"])
    ap.add_argument("--grid", type=int, default=0)
    ap.add_argument("--serial", action="store_true", help="one wave at a time: offload, then restore (no duplex overlap)")
    ap.add_argument("--wave-frac", type=int, default=8, help="pipelined schedule: a wave uses 1/N of the pool (N >= 2)")
    ap.add_argument("--dedup", action="store_true", help="NEXT-2: content-addressed host store; value counts claim-logical bytes")
    ap.add_argument("--direct-offload", action="store_true", help="NEXT-4 experiment: gather straight into the mapped pinned store")
    ap.add_argument("--layer-major", action="store_true", help="NEXT-4: layer-major host copy and streaming order")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--per-config-budget-s", type=float, default=270.0,
                    help="wall-clock budget for the per_config block (the other four configs, 3 steps each); 0 = off")
    ap.add_argument("--traffic", type=float, default=None, help="ncu dram bytes per gather launch (profiles/), if known")
    a = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    wname = "configs[%d] %s" % (a.config, W.GEOMS[a.config].name)

    if a.impl == "reference":
        if rank != 0:
            return
        steps, warmup = max(1, min(a.steps, 3)), min(a.warmup, 1)
        res = run_oracle(a.config, steps, warmup)
        line = {"impl": "reference", "metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": a.gpus,
                "steps": steps, "warmup": warmup, "ms_per_step": res["seconds"] * 1e3 / steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
                "config": {"workload": wname, "sample": res["sample"]}, "claims_per_s": res["claims_per_s"],
                "cpu_baseline": {"value": res["value"], "unit": UNIT, "cores": 1, "kind": "oracle", "sample": res["sample"]},
                "e2e": {"value": res["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line))
        return

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; librc has no CPU path (use --impl reference for the oracle)")
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2606_01387_b200 import rc, tp
    numa = tp.bind_to_gpu_numa_node(local)      # before rc_create: the pinned store is first touched on the GPU's node
    mover = {"auto": rc.MOVER_AUTO, "ldg": rc.MOVER_LDG, "tma": rc.MOVER_TMA}[a.mover]
    job = Job(a.config, rank, world, a.chunk_mib << 20, mover, a.grid, pipelined=not a.serial, wave_frac=max(2, a.wave_frac), dedup=a.dedup, direct=a.direct_offload,
              layer_major=a.layer_major)
    g = job.g
    link = {}

    def measure_ceilings():
        # pinned-copy ceilings of this process (the store holds no claim bytes between steps); the best of the
        # measurements taken before and after the timed region counts: the first copies on a fresh box run slow
        for name, d in (("d2h", 0), ("h2d", 1), ("both", 2)):
            link[name] = max(link.get(name, 0.0), job.r.measure_link(1 << 30, d, reps=6))
    if world == 1:
        measure_ceilings()

    sampler = ClockSampler(local) if rank == 0 else None
    ms, wall_ms, st = time_steps(job, a.steps, a.warmup, False, dist)
    clocks = sampler.stop() if sampler else None
    if world == 1:
        measure_ceilings()
    payload = st["bytes_d2h"] + st["bytes_h2d"]
    link_bytes = payload
    if a.dedup:                # claim-logical bytes moved (what the claims hold), not the smaller number that crossed the link
        payload = (st["gather_blocks"] + st["scatter_blocks"]) * job.g.blk_bytes
    claims = sum(p["n"] for p in job.prep) * a.steps
    e2e = None
    if not a.no_e2e:
        ms2, _, st2 = time_steps(job, a.steps, min(a.warmup, 1), True, dist)
        e2e = (ms2, st2)

    ms_max = reduce_scalar(dist, ms, "max")
    payload_all = reduce_scalar(dist, float(payload), "sum")
    claims_all = reduce_scalar(dist, float(claims), "sum")
    launches_all = reduce_scalar(dist, float(st["kernel_launches"]), "sum")
    if e2e:
        ms2_max = reduce_scalar(dist, e2e[0], "max")
        pay2_all = reduce_scalar(dist, float(e2e[1]["bytes_d2h"] + e2e[1]["bytes_h2d"]), "sum")
    if rank != 0:
        dist.destroy_process_group()
        return

    peak, peak_src = peaks()
    blk = g.blk_bytes

    def roof(ms_k, launches, blocks):
        if not launches or ms_k <= 0:
            return None
        per_launch = 2.0 * blk * blocks / launches                  # algorithmic bytes: read blk + write blk per block
        ach = per_launch / (ms_k / launches * 1e6)
        return {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "traffic": a.traffic, "peak_source": peak_src, "launches": launches,
                "avg_launch_ms": ms_k / launches, "algorithmic_bytes_per_launch": per_launch}

    traffic_source = "--traffic" if a.traffic is not None else None
    if a.traffic is None:      # dram__bytes_read+write of the gather kernel from the committed ncu capture, scaled per block
        try:
            with open(os.path.join(ROOT, "profiles", "r02_traffic.json")) as f:
                tj = json.load(f)
            a.traffic = (tj["dram_bytes_read"] + tj["dram_bytes_write"]) / tj["launch_blocks"] * st["gather_blocks"] / max(1, st["gather_launches"])
            traffic_source = "profiles/r02_traffic.json: " + tj["source"] + "; scaled by blocks per launch (not measured in this run: ncu is needed)"
        except Exception:
            a.traffic = None
    roofline = roof(st["ms_gather"], st["gather_launches"], st["gather_blocks"])
    if roofline:
        roofline["kernel"] = "k_move_hash%s<GATHER> (K2 gather+checksum)" % ("_tma" if mover != rc.MOVER_LDG else "")
        roofline["traffic_source"] = traffic_source
        roofline["note"] = ("measured inside the pipelined step, both copy engines active; the same kernel alone on the device: "
                            "0.97-0.99 by CUDA events, 1.01-1.03 by ncu (profiles/r02_mover_sweep.md, r02_prof_c1.md, r02_instep_trace.md)")
    roof_sc = roof(st["ms_scatter"], st["scatter_launches"], st["scatter_blocks"])
    if roof_sc:
        roof_sc["kernel"] = "k_move_hash%s<SCATTER> (K4 scatter+checksum)" % ("_tma" if mover != rc.MOVER_LDG else "")
        roof_sc["traffic"] = None
        roof_sc["note"] = ("measured inside the pipelined step; since the restore's last chunk is cut the main scatter runs beside "
                           "both copy engines (DESIGN.md 6); alone on the device: 0.99-1.00")
    roof_dg = None
    if world == 1:             # M3: the checksum alone, read-only pass over one staging-sized buffer (algorithmic bytes = blk per block)
        nblk = int(min(a.chunk_mib << 20, job.host_store) // blk)
        buf = torch.empty(nblk * blk, dtype=torch.uint8, device="cuda")
        buf.random_(0, 256)
        torch.cuda.synchronize()
        best = None
        for _ in range(4):
            _, ms_d = job.r.digest_blocks(buf.data_ptr(), nblk, want=False)
            best = ms_d if best is None else min(best, ms_d)
        ach = nblk * blk / (best * 1e6)
        roof_dg = {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": None,
                   "kernel": "k_move_hash_tma<DIGEST> (checksum only, read-only)", "launch_ms": best,
                   "algorithmic_bytes_per_launch": nblk * blk, "note": "read-only stream against a copy-rate peak (read+write)"}
        del buf
    links = None
    if link:
        d2h = st["bytes_d2h"] / (st["ms_d2h"] * 1e6) if st["ms_d2h"] > 0 else None
        h2d = st["bytes_h2d"] / (st["ms_h2d"] * 1e6) if st["ms_h2d"] > 0 else None
        links = {"ceiling_gbs": link, "d2h_gbs": d2h, "h2d_gbs": h2d,
                 "d2h_frac": d2h / link["d2h"] if d2h else None, "h2d_frac": h2d / link["h2d"] if h2d else None,
                 "ceiling_how": "best of 2 x 6 cudaMemcpyAsync of 1 GiB (before and after the timed region), pinned store <-> staging, same process; "
                                "'both' = D2H and H2D at once (sum); fractions are per direction over that "
                                "direction's copy-stream busy time against its one-way ceiling"}
    line = {"metric": METRIC, "value": payload_all / (ms_max * 1e6), "unit": UNIT, "n_gpus": world, "steps": a.steps,
            "warmup": a.warmup, "ms_per_step": ms_max / a.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u8", "data": "synthetic",
            "config": {"workload": wname, "claims": len(job.wl.claims), "pool_blocks": g.pool_blocks, "blk_bytes": blk,
                       "waves": len(job.waves), "host_store_bytes": job.host_store, "staging_chunk_bytes": a.chunk_mib << 20,
                       "mover": a.mover, "schedule": "serial" if a.serial else "restore(k) overlapped with offload(k+1) and offload(k+2) (two open offloads); waves of consecutive steps form one sequence", "l2": "inputs larger than L2 (pool %d GiB, staging chunks %d MiB, L2 126 MB)" % (g.pool_bytes >> 30, a.chunk_mib),
                       "parallelism": "claims independent: one replica of the workload per GPU, no collective",
                       "numa_node": numa, "layer_major": bool(a.layer_major)},
            "claims_per_s": claims_all / (ms_max / 1e3), "payload_bytes_per_step": payload_all / a.steps,
            "wall_ms_per_step": wall_ms / a.steps, "clocks": clocks, "gpu_launches": int(launches_all),
            "dedup": ({"link_bytes_per_step": link_bytes / a.steps, "logical_bytes_per_step": payload / a.steps,
                       "link_over_logical": link_bytes / max(1, payload)} if a.dedup else None),
            "roofline": roofline, "roofline_scatter": roof_sc, "roofline_digest": roof_dg, "host_link": links}
    if links:
        links["value_over_duplex_ceiling"] = line["value"] / link["both"]
    if e2e:
        n_ev = job.events
        line["e2e"] = {"value": pay2_all / (ms2_max * 1e6), "unit": UNIT,
                       "h2d_bytes_per_step": int(e2e[1]["bytes_h2d"] / a.steps + job.meta_h2d + job.fill_h2d),
                       "d2h_bytes_per_step": int(e2e[1]["bytes_d2h"] / a.steps + 32 * n_ev + 4 * 5 * claims / a.steps),
                       "ms_per_step": ms2_max / a.steps,
                       "what": "same step through the C ABI with host arrays; fill[] sent as host arrays (rc_set_fill), "
                               "statuses and the event stream read back, inside the timed region"}
    if world == 1:
        try:
            line["single_claim"] = single_claim_latency(job)
        except Exception as e:                                                 # a side measurement must not lose the main line
            line["single_claim"] = {"error": repr(e)[:200]}
    if world == 1 and not a.no_cpu_baseline:   # NEXT-1: device trace validator on a 200k-claim synthetic stream (not part of `value`)
        sys.path.insert(0, os.path.join(ROOT, "tests"))
        import trace_inputs                                  # input generator only (tests/trace_inputs.py)
        tr = trace_inputs.make_trace(200000, 1)
        best = None
        for _ in range(3):
            rep, _c = rc.validate_trace(tr, want_claims=False)
            best = rep if best is None or rep["ms_kernels"] < best["ms_kernels"] else best
        line["trace_validator"] = {"events": int(tr.size), "claims": int(best["n_claims"]), "ok": int(best["ok"]),
                                   "ms_kernels": best["ms_kernels"], "ms_with_copies": best["ms_total"],
                                   "events_per_s_kernels": tr.size / (best["ms_kernels"] * 1e-3)}
    if world == 1 and not a.no_cpu_baseline:
        line["cpu_baseline"] = {k: v for k, v in run_oracle(a.config, 1, 0).items() if k in
                                ("value", "unit", "cores", "kind", "sample", "claims_per_s", "seconds")}
        line["cpu_baseline"]["all_cores"] = run_oracle_all_cores(a.config)
    if world == 1 and a.per_config_budget_s > 0:
        # the other BASELINE.json configs at full size, same schedule, >= 3 steps each, device-timed like `value`;
        # a config whose estimated cost does not fit the remaining budget is skipped and says so
        job.close()
        t_start = time.perf_counter()
        per = {"configs[%d]" % a.config: {"value": line["value"], "claims_per_s": line["claims_per_s"], "steps": a.steps,
                                          "ms_per_step": line["ms_per_step"], "gather_frac": roofline and roofline["frac"],
                                          "scatter_frac": roof_sc and roof_sc["frac"],
                                          "value_over_duplex_ceiling": links and links.get("value_over_duplex_ceiling")}}
        for idx in (3, 0, 4, 2):
            if idx == a.config:
                continue
            wl_i = W.make_workload(idx)
            est_bytes = 2.0 * sum(((c.M + wl_i.geom.block_size - 1) // wl_i.geom.block_size) * wl_i.geom.blk_bytes
                                  for c in wl_i.claims if c.M >= c.N)
            est_step = est_bytes / 85e9
            wu = 1 if est_step < 5 else 0            # a step of many seconds is its own warm-up (this block is a side measurement)
            est = (3 + wu) * est_step + 15 + wl_i.geom.pool_bytes / 4e9       # warm-up + 3 steps, setup, pool generation
            left = a.per_config_budget_s - (time.perf_counter() - t_start)
            key = "configs[%d] %s" % (idx, W.GEOMS[idx].name)
            if est > left:
                per[key] = {"skipped": "estimated %.0f s, %.0f s of the budget left (run: python bench.py --config %d)" % (est, left, idx)}
                continue
            try:
                j2 = Job(idx, rank, world, a.chunk_mib << 20, mover, a.grid, pipelined=not a.serial, wave_frac=max(2, a.wave_frac))
                ms_i, _, st_i = time_steps(j2, 3, wu, False, None)
                pay = st_i["bytes_d2h"] + st_i["bytes_h2d"]
                blk_i = j2.g.blk_bytes

                def fr(ms_k, launches, blocks):
                    return (2.0 * blk_i * blocks / (ms_k * 1e6)) / peak if launches and ms_k > 0 else None
                per[key] = {"value": pay / (ms_i * 1e6), "claims_per_s": sum(p["n"] for p in j2.prep) * 3 / (ms_i / 1e3),
                            "steps": 3, "warmup": wu, "ms_per_step": ms_i / 3, "waves": len(j2.waves),
                            "payload_bytes_per_step": pay / 3, "pool_blocks": j2.g.pool_blocks,
                            "gather_frac": fr(st_i["ms_gather"], st_i["gather_launches"], st_i["gather_blocks"]),
                            "scatter_frac": fr(st_i["ms_scatter"], st_i["scatter_launches"], st_i["scatter_blocks"]),
                            "d2h_gbs": st_i["bytes_d2h"] / (st_i["ms_d2h"] * 1e6) if st_i["ms_d2h"] > 0 else None,
                            "h2d_gbs": st_i["bytes_h2d"] / (st_i["ms_h2d"] * 1e6) if st_i["ms_h2d"] > 0 else None,
                            "value_over_duplex_ceiling": pay / (ms_i * 1e6) / link["both"] if link else None,
                            "gpu_launches": int(st_i["kernel_launches"])}
                j2.close()
            except Exception as e:                                             # a side measurement must not lose the main line
                per[key] = {"error": repr(e)[:200]}
        line["per_config"] = per
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
