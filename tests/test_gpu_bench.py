"""bench.py's own step on the GPU at the smallest config: the pipelined schedule (two open offloads), its dedup form (one
open offload), the layer-major option and the serial schedule all drive the library without a refused call, move every
claim once per direction per step, and leave a stream the oracle's validator accepts."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import bench
from oracle import validator as V
from paper_2606_01387_b200 import rc


@pytest.mark.parametrize("mode", ["pipelined", "dedup", "layer_major", "serial"])
def test_bench_step_on_tiny(mode):
    job = bench.Job(0, 0, 1, 1 << 20, rc.MOVER_AUTO, 0, pipelined=mode != "serial", wave_frac=8,
                    dedup=mode == "dedup", layer_major=mode == "layer_major")
    events = []
    real_outcomes = job.r.outcomes

    def tap(cap=1 << 20):
        ev = real_outcomes(cap=cap)
        events.append(ev)
        return ev
    job.r.outcomes = tap
    ms, wall, st = bench.time_steps(job, 2, 1, False, None)     # raises if a claim was skipped (consistency check)
    want = sum(1 for c in job.wl.claims if c.M >= c.N) * 2
    assert st["claims_offloaded"] == want and st["claims_restored"] + st["claims_refused"] == want
    assert st["claims_refused"] == 2 * sum(1 for c in job.wl.claims if c.fault)
    assert st["gather_launches"] > 0 and st["scatter_launches"] > 0 and ms > 0
    ev = np.concatenate(events)
    assert list(ev["seq"]) == list(range(int(ev["seq"][0]), int(ev["seq"][0]) + len(ev)))
    # claim ids recur from step to step (accept ... release, accept ...): every acceptance starts a new claim for the validator
    ev = ev.copy()
    n_accepts, alias = {}, {}
    for e in ev:
        cid = int(e["claim_id"])
        if int(e["code"]) == 1:
            n_accepts[cid] = n_accepts.get(cid, 0) + 1
            alias[cid] = (cid ^ (n_accepts[cid] << 48)) | 1
        if int(e["code"]) == 8 and int(e["aux"]) == 1:
            e["arg"] = alias[cid]                                  # blocking_claim_ids = [C]
        e["claim_id"] = alias[cid]
    ok, why = V.validate(ev)
    assert ok, why
    job.close()


def test_bench_line_contract_on_tiny():
    """`python bench.py` prints ONE JSON line with the keys the driver reads (smallest config, seconds)."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--config", "0", "--steps", "3", "--warmup", "3",
                          "--no-cpu-baseline", "--per-config-budget-s", "0"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    l = json.loads(lines[0])
    assert l["metric"] == "kv_offload_restore_throughput" and l["unit"] == "GB/s" and l["higher_is_better"] is True
    assert l["n_gpus"] == 1 and l["steps"] == 3 and l["warmup"] == 3 and l["scaling"] == "weak" and l["vs_baseline"] is None
    assert l["dtype"] == "u8" and l["data"] == "synthetic" and l["config"]["workload"].startswith("configs[0]")
    assert l["value"] > 0 and l["ms_per_step"] > 0 and l["gpu_launches"] > 0
    r = l["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9 and "traffic" in r
    e = l["e2e"]
    assert e["value"] > 0 and e["unit"] == "GB/s" and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    assert set(l["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    assert l["single_claim"]["restore_ms"] > 0
