"""Multi-GPU plumbing around librc: argument marshalling and torch.distributed calls only.

(1) Claim-sharded replicas -- each GPU owns a pool, a pinned store and a host link; no data-path collective:
    `merge_outcomes` joins the per-GPU outcome streams on the host by (gpu, seq); `bind_to_gpu_numa_node` keeps the
    process (and therefore the first-touch pages of the pinned store) on the GPU's NUMA node.
(2) TP-sharded KV -- the pool is split by kv_head over G ranks; every rank makes the same calls on its shard.  The
    restoration verdict must be common, so between rc_tp_restore_verify and rc_tp_restore_commit the ranks exchange
    8-byte verdict records per claim: `all_gather_verdicts` (one all-gather: NCCL on device tensors, gloo on CPU
    tensors), or -- on NVLink / NVSwitch -- peer mailboxes that the verify step writes directly (`open_peer_mailboxes`),
    with one barrier instead of a collective.  The merge itself (AND of ok, min of the failing block index) runs in the
    library's k_tp_merge kernel, never here.
"""
import ctypes as C
import os

import numpy as np

VERDICT_DTYPE = np.dtype([("flags", "<u4"), ("bad", "<u4")])          # flags: 1 = served, 2 = locally ok
V_SERVED, V_OK = 1, 2


def shard_kv_heads(pool, layers, pool_blocks, block_size, kv_heads, head_dim, elem_bytes, rank, ranks):
    """The kv_head shard `rank` of a full pool laid out [L][2][NB][BS][H][D]: heads rank*H/G .. (rank+1)*H/G.
    Works on numpy arrays and torch tensors of bytes; returns a contiguous copy in the same layout with H/G heads."""
    assert kv_heads % ranks == 0
    hs = kv_heads // ranks
    v = pool.reshape(layers, 2, pool_blocks, block_size, kv_heads, head_dim * elem_bytes)
    part = v[:, :, :, :, rank * hs:(rank + 1) * hs, :]
    return (part.contiguous() if hasattr(part, "contiguous") else np.ascontiguousarray(part)).reshape(-1)


def all_gather_verdicts(local, dist=None, device="cpu"):
    """[n] local verdict records -> [G, n] records of all ranks, rank-major.  One all-gather of 8 bytes per claim;
    `device` "cpu" for gloo, a CUDA device for NCCL.  Without a process group: G = 1."""
    local = np.ascontiguousarray(local, dtype=VERDICT_DTYPE)
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local.reshape(1, -1).copy()
    import torch
    t = torch.from_numpy(local.view(np.uint8).copy()).to(device)
    out = [torch.empty_like(t) for _ in range(dist.get_world_size())]
    dist.all_gather(out, t)
    return np.stack([o.cpu().numpy().view(VERDICT_DTYPE) for o in out])


def tp_restore(r, claim_ids, dist=None, device="cpu"):
    """A TP-sharded restore on one rank through the all-gather path: verify (a5-a7 on this rank's shard), exchange,
    commit (merge in k_tp_merge, a8).  Every rank calls this with the same ids.  Returns the statuses."""
    st, local = r.tp_restore_verify(claim_ids)
    return r.tp_restore_commit(all_gather_verdicts(local, dist, device), st)


def open_peer_mailboxes(r, dist):
    """NVLink path: exchanges the CUDA IPC handles of the ranks' verdict mailboxes (one all_gather_object at set-up) and
    opens the peers' mailboxes, after which rc_tp_restore_verify writes this rank's records straight into every peer's
    mailbox and a barrier replaces the collective: tp_restore_mailbox."""
    handles = [None] * dist.get_world_size()
    dist.all_gather_object(handles, r.tp_ipc_handle())
    for rank, h in enumerate(handles):
        if rank != dist.get_rank():
            r.tp_open_peer(rank, h)


def tp_restore_mailbox(r, claim_ids, dist):
    st, _ = r.tp_restore_verify(claim_ids)
    dist.barrier()                                         # every rank's verify (and its peer stores) has completed
    return r.tp_restore_commit(None, st)


def merge_outcomes(streams):
    """Claim-sharded replicas: per-GPU outcome streams (each in its own seq order) -> one stream ordered by (gpu, seq),
    renumbered 0.. in that order; `origin` keeps (gpu, original seq) per record.  A claim lives on one GPU, so its
    records stay contiguous in their own order and attribution survives the merge."""
    dt = streams[0].dtype if streams else None
    merged = np.concatenate([np.asarray(s) for s in streams]) if streams else np.zeros(0, dt)
    origin = np.zeros(merged.size, np.dtype([("gpu", "<u4"), ("seq", "<u8")]))
    at = 0
    for g, s in enumerate(streams):
        assert s.size == 0 or (np.diff(s["seq"].astype(np.int64)) > 0).all(), "per-GPU stream must be in seq order"
        origin["gpu"][at:at + s.size] = g
        origin["seq"][at:at + s.size] = s["seq"]
        at += s.size
    merged = merged.copy()
    merged["seq"] = np.arange(merged.size, dtype=np.uint64)
    return merged, origin


def gpu_numa_node(local_rank=0):
    """NUMA node of the GPU (sysfs), or None when the platform does not say (single-socket boxes report -1)."""
    try:
        import torch
        bus = torch.cuda.get_device_properties(local_rank).pci_bus_id if hasattr(
            torch.cuda.get_device_properties(local_rank), "pci_bus_id") else None
        dom = getattr(torch.cuda.get_device_properties(local_rank), "pci_domain_id", 0)
        dev = getattr(torch.cuda.get_device_properties(local_rank), "pci_device_id", 0)
        if bus is None:
            return None
        path = "/sys/bus/pci/devices/%04x:%02x:%02x.0/numa_node" % (dom, bus, dev)
        node = int(open(path).read().strip())
        return node if node >= 0 else None
    except Exception:
        return None


def parse_cpulist(text):
    cpus = set()
    for part in text.strip().split(","):
        if not part:
            continue
        lo, _, hi = part.partition("-")
        cpus.update(range(int(lo), int(hi or lo) + 1))
    return cpus


def bind_to_gpu_numa_node(local_rank=0):
    """Pins this process to the CPUs of the GPU's NUMA node BEFORE the context is created, so that the pinned host
    store (cudaHostAlloc, first touch under the default local policy) and the submitting thread sit next to the
    GPU's PCIe root.  Returns the node, or None if nothing was changed."""
    node = gpu_numa_node(local_rank)
    if node is None or not hasattr(os, "sched_setaffinity"):
        return None
    try:
        cpus = parse_cpulist(open("/sys/devices/system/node/node%d/cpulist" % node).read())
        cpus &= os.sched_getaffinity(0)
        if cpus:
            os.sched_setaffinity(0, cpus)
            return node
    except Exception:
        pass
    return None
