import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has = torch.cuda.is_available()
    except Exception:
        has = False
    if has:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)


def build_tiny_oracle(wl=None, host_store_bytes=1 << 40, poison=True):
    """Tiny config on the oracle: returns (oracle, workload, wave, pool, fill)."""
    from oracle import rco
    from paper_2606_01387_b200 import workloads as W
    wl = wl or W.make_workload(0)
    g = wl.geom
    wave = W.plan_waves(wl, host_store_bytes)[0]
    pool = W.pool_host(g)
    fill = np.zeros(g.pool_blocks, np.uint8)
    fill[wave.fill_ids] = wave.fill_val
    o = rco.Oracle(g.layers, g.kv_heads, g.head_dim, g.elem_bytes, g.block_size, g.pool_blocks, pool, fill,
                   host_store_bytes)
    o.mark_used(wave.used_ids)
    return o, wl, wave, pool, fill
