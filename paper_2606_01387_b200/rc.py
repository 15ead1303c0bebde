"""ctypes binding over librc.so (include/rc.h): argument marshalling only.

Every step of the path runs inside the library's sm_100a kernels; this module converts numpy
arrays to pointers and back.  PyTorch supplies the device memory (pool, fill) and, optionally,
the CUDA streams.  Importing this module builds/loads the CUDA extension and fails loudly if
that is impossible -- there is no CPU fallback.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

EVENT_DTYPE = np.dtype([("seq", "<u8"), ("claim_id", "<u8"), ("code", "<u4"), ("aux", "<u4"), ("arg", "<u8")])
FAULT_DTYPE = np.dtype([("claim_id", "<u8"), ("kind", "<u4"), ("param", "<u4")])
TP_VERDICT_DTYPE = np.dtype([("flags", "<u4"), ("bad", "<u4")])      # rc_tp_verdict: flags 1 = served, 2 = locally ok

OK, ERR_INVALID, ERR_CUDA, ERR_NOMEM, ERR_CAPACITY, ERR_BUSY = 0, -1, -2, -3, -4, -5
ST_OK, ST_PRED_FALSE, ST_UNKNOWN_CLAIM, ST_BAD_STATE, ST_DUPLICATE_ID, ST_BAD_TABLE = 0, 1, 2, 3, 4, 5
ST_NO_FREE_BLOCKS, ST_NO_HOST_SPACE, ST_RESTORE_FAILED, ST_PROTECTED_CONFLICT = 6, 7, 8, 9
FAULT_XFER_ERROR, FAULT_BITFLIP, FAULT_ALLOW_UNCLAIMED = 1, 2, 1
MOVER_AUTO, MOVER_LDG, MOVER_TMA = 0, 1, 2
REQ_FLAG = 0x80000000
POLICY_REFUSE, POLICY_DEMOTE, POLICY_EXPIRE = 0, 1, 2

EXPORTS = ["rc_create", "rc_destroy", "rc_mark_used", "rc_mark_free", "rc_set_fill", "rc_accept", "rc_materialize", "rc_offload",
           "rc_restore", "rc_offload_begin", "rc_restore_begin", "rc_wait", "rc_test", "rc_set_policy", "rc_restore_request",
           "rc_restore_request_begin", "rc_tp_restore_verify", "rc_tp_restore_commit", "rc_tp_mailbox", "rc_tp_set_peer",
           "rc_tp_ipc_handle", "rc_tp_open_peer", "rc_protect", "rc_make_room", "rc_protected_map", "rc_outcomes", "rc_set_faults",
           "rc_release", "rc_claim_info", "rc_claim_blocks", "rc_claim_digests", "rc_host_read", "rc_host_store", "rc_sync", "rc_pool_state",
           "rc_stats_get", "rc_stats_reset", "rc_measure_link", "rc_digest_blocks", "rc_digest_blocks_noalloc", "rc_validate_trace", "rc_strerror",
           "rc_last_cuda_error"]


class Config(C.Structure):
    _fields_ = [("layers", C.c_uint32), ("kv_heads", C.c_uint32), ("head_dim", C.c_uint32), ("elem_bytes", C.c_uint32),
                ("block_size", C.c_uint32), ("pool_blocks", C.c_uint32), ("max_claims", C.c_uint32),
                ("max_table_entries", C.c_uint32), ("max_events", C.c_uint32), ("staging_chunks", C.c_uint32),
                ("staging_chunk_bytes", C.c_uint64), ("host_store_bytes", C.c_uint64),
                ("pool_dev", C.c_void_p), ("fill_dev", C.c_void_p),
                ("stream_meta", C.c_void_p), ("stream_gather", C.c_void_p), ("stream_d2h", C.c_void_p),
                ("stream_scatter", C.c_void_p), ("stream_h2d", C.c_void_p),
                ("mover", C.c_uint32), ("grid_ctas", C.c_uint32), ("dedup", C.c_uint32), ("direct_offload", C.c_uint32),
                ("tp_ranks", C.c_uint32), ("tp_rank", C.c_uint32), ("layer_major", C.c_uint32)]


class ClaimInfo(C.Structure):
    _fields_ = [("claim_id", C.c_uint64), ("chain", C.c_uint64), ("host_bytes", C.c_uint64),
                ("state", C.c_uint32), ("P", C.c_uint32), ("N", C.c_uint32), ("M", C.c_uint32),
                ("nb", C.c_uint32), ("n_table", C.c_uint32)]


class Stats(C.Structure):
    _fields_ = [("bytes_d2h", C.c_uint64), ("bytes_h2d", C.c_uint64), ("claims_offloaded", C.c_uint64),
                ("claims_restored", C.c_uint64), ("claims_refused", C.c_uint64), ("generic_failures", C.c_uint64),
                ("host_used_bytes", C.c_uint64), ("free_blocks", C.c_uint64), ("events_emitted", C.c_uint64),
                ("kernel_launches", C.c_uint64), ("ms_gather", C.c_float), ("ms_scatter", C.c_float),
                ("ms_d2h", C.c_float), ("ms_h2d", C.c_float), ("gather_launches", C.c_uint64),
                ("scatter_launches", C.c_uint64), ("gather_blocks", C.c_uint64), ("scatter_blocks", C.c_uint64)]


class TraceReport(C.Structure):
    _fields_ = [("first_bad_index", C.c_uint64), ("n_events", C.c_uint64), ("n_claims", C.c_uint64),
                ("n_failure_gate", C.c_uint64), ("n_observation_gate", C.c_uint64), ("ok", C.c_uint32), ("pad", C.c_uint32),
                ("ms_kernels", C.c_float), ("ms_total", C.c_float)]


TRACE_CLAIM_DTYPE = np.dtype([("claim_id", "<u8"), ("first_bad", "<u8"), ("state", "<u4"), ("gates", "<u4"),
                              ("n_events", "<u4"), ("pad", "<u4")])
GATE_FAILURE, GATE_OBSERVATION = 1, 2
NO_BAD = (1 << 64) - 1

_lib = None


def lib():
    """Loads librc.so, building it in-tree first if a source is newer.  Raises if it cannot."""
    global _lib
    if _lib is None:
        so = _build.SO if os.environ.get("RC_NO_BUILD") and os.path.exists(_build.SO) else _build.build()
        _lib = C.CDLL(so)
        _lib.rc_strerror.restype = C.c_char_p
        _lib.rc_last_cuda_error.restype = C.c_char_p
        _lib.rc_last_cuda_error.argtypes = [C.c_void_p]
    return _lib


class RcError(RuntimeError):
    def __init__(self, code, what, detail=""):
        super().__init__("%s: %d (%s) %s" % (what, code, lib().rc_strerror(code).decode(), detail))
        self.code = code


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _u64(x):
    return np.ascontiguousarray(x, dtype=np.uint64)


def _u32(x):
    return np.ascontiguousarray(x, dtype=np.uint32)


class RC:
    """One librc context over a caller-owned device pool and fill vector (torch uint8 tensors)."""

    def __init__(self, layers, kv_heads, head_dim, elem_bytes, block_size, pool_blocks, pool, fill,
                 host_store_bytes, staging_chunk_bytes=None, staging_chunks=2, max_claims=8192,
                 max_table_entries=None, max_events=1 << 17, streams=None, mover=MOVER_AUTO, grid_ctas=0, dedup=False, direct_offload=False,
                 tp_ranks=0, tp_rank=0, layer_major=False):
        self.L = lib()
        page = block_size * kv_heads * head_dim * elem_bytes
        self.page, self.blk, self.NB = page, 2 * layers * page, pool_blocks
        assert pool.is_cuda and fill.is_cuda, "librc needs device memory: there is no CPU path"
        assert pool.numel() * pool.element_size() == self.blk * pool_blocks and fill.numel() == pool_blocks
        self.pool, self.fill = pool, fill                      # keep the tensors alive
        self.streams = streams
        s = [0] * 5 if streams is None else [int(x.cuda_stream) for x in streams]
        cfg = Config(layers, kv_heads, head_dim, elem_bytes, block_size, pool_blocks, max_claims,
                     max_table_entries or max(4 * pool_blocks, 1 << 16), max_events, staging_chunks,
                     staging_chunk_bytes or min(1 << 30, max(self.blk, host_store_bytes)), host_store_bytes,
                     pool.data_ptr(), fill.data_ptr(), s[0], s[1], s[2], s[3], s[4], mover, grid_ctas, int(dedup), int(direct_offload), tp_ranks, tp_rank, int(layer_major))
        self.tp_ranks = max(1, tp_ranks)
        self.h = C.c_void_p()
        rc = self.L.rc_create(C.byref(cfg), C.byref(self.h))
        if rc != 0:
            self.h = None
            raise RcError(rc, "rc_create")
        self._pending = {}

    def close(self):
        if getattr(self, "h", None):
            self.L.rc_destroy(self.h)
            self.h = None
        self.pool = self.fill = None                           # the caller's tensors are no longer needed

    def __del__(self):
        self.close()

    def _ck(self, rc, what):
        if rc != 0:
            raise RcError(rc, what, self.L.rc_last_cuda_error(self.h).decode())

    def mark_used(self, ids):
        ids = _u32(ids)
        return self.L.rc_mark_used(self.h, ids.size, _p(ids))

    def set_fill(self, ids, vals):
        ids, vals = _u32(ids), np.ascontiguousarray(vals, dtype=np.uint8)
        assert ids.size == vals.size
        self._ck(self.L.rc_set_fill(self.h, ids.size, _p(ids), _p(vals)), "rc_set_fill")

    def mark_free(self, ids):
        ids = _u32(ids)
        return self.L.rc_mark_free(self.h, ids.size, _p(ids))

    def accept(self, claim_ids, P, N, bt_off, bt_ids, check=True):
        claim_ids, P, N, bt_off, bt_ids = _u64(claim_ids), _u32(P), _u32(N), _u32(bt_off), _u32(bt_ids)
        st = np.full(claim_ids.size, -1, np.int32)
        rc = self.L.rc_accept(self.h, claim_ids.size, _p(claim_ids), _p(P), _p(N), _p(bt_off), _p(bt_ids), _p(st))
        if check:
            self._ck(rc, "rc_accept")
            return st
        return rc, st

    def _batch(self, fn, name, claim_ids, check=True):
        claim_ids = _u64(claim_ids)
        st = np.full(claim_ids.size, -1, np.int32)
        rc = fn(self.h, claim_ids.size, _p(claim_ids), _p(st))
        if check:
            self._ck(rc, name)
            return st
        return rc, st

    def materialize(self, ids, **kw):
        return self._batch(self.L.rc_materialize, "rc_materialize", ids, **kw)

    def offload(self, ids, **kw):
        return self._batch(self.L.rc_offload, "rc_offload", ids, **kw)

    def restore(self, ids, **kw):
        return self._batch(self.L.rc_restore, "rc_restore", ids, **kw)

    def release(self, ids, **kw):
        return self._batch(self.L.rc_release, "rc_release", ids, **kw)

    def offload_begin(self, ids):
        ids = _u64(ids)
        st = np.full(ids.size, -1, np.int32)
        self._ck(self.L.rc_offload_begin(self.h, ids.size, _p(ids), _p(st)), "rc_offload_begin")
        # every _begin is paired with one wait(); served entries are pending (-1) iff the library opened an operation
        self._pending.setdefault(0, []).append((ids, st, bool((st == -1).any())))
        return st

    def restore_begin(self, ids):
        ids = _u64(ids)
        st = np.full(ids.size, -1, np.int32)
        self._ck(self.L.rc_restore_begin(self.h, ids.size, _p(ids), _p(st)), "rc_restore_begin")
        self._pending.setdefault(1, []).append((ids, st, bool((st == -1).any())))
        return st

    def restore_request(self, request_id, ids, check=True):
        ids = _u64(ids)
        st = np.full(ids.size, -1, np.int32)
        rc = self.L.rc_restore_request(self.h, C.c_uint64(request_id), ids.size, _p(ids), _p(st))
        if check:
            self._ck(rc, "rc_restore_request")
            return st
        return rc, st

    def restore_request_begin(self, request_id, ids):
        ids = _u64(ids)
        st = np.full(ids.size, -1, np.int32)
        self._ck(self.L.rc_restore_request_begin(self.h, C.c_uint64(request_id), ids.size, _p(ids), _p(st)),
                 "rc_restore_request_begin")
        self._pending.setdefault(1, []).append((ids, st, bool((st == -1).any())))
        return st

    def set_policy(self, ids, policy):
        ids, policy = _u64(ids), _u32(policy)
        return self.L.rc_set_policy(self.h, ids.size, _p(ids), _p(policy))

    def tp_restore_verify(self, ids):
        """Phase 1 of a TP-sharded restore (rc.h): returns (statuses, local verdict records)."""
        ids = _u64(ids)
        st = np.full(ids.size, -1, np.int32)
        v = np.zeros(ids.size, TP_VERDICT_DTYPE)
        self._ck(self.L.rc_tp_restore_verify(self.h, ids.size, _p(ids), _p(st), _p(v)), "rc_tp_restore_verify")
        return st, v

    def tp_restore_commit(self, gathered, st, check=True):
        """Phase 2: gathered = [ranks, n] records of all ranks, or None to read this rank's peer mailbox."""
        if gathered is None:
            rc = self.L.rc_tp_restore_commit(self.h, st.size, self.tp_ranks, None, _p(st))
        else:
            g = np.ascontiguousarray(gathered, dtype=TP_VERDICT_DTYPE)
            assert g.ndim == 2
            rc = self.L.rc_tp_restore_commit(self.h, g.shape[1], g.shape[0], _p(g), _p(st))
        if check:
            self._ck(rc, "rc_tp_restore_commit")
            return st
        return rc, st

    def tp_mailbox(self):
        p, n = C.c_void_p(), C.c_uint64()
        self._ck(self.L.rc_tp_mailbox(self.h, C.byref(p), C.byref(n)), "rc_tp_mailbox")
        return p.value, n.value

    def tp_set_peer(self, rank, mailbox_ptr):
        return self.L.rc_tp_set_peer(self.h, rank, C.c_void_p(mailbox_ptr))

    def tp_ipc_handle(self):
        buf = C.create_string_buffer(64)
        self._ck(self.L.rc_tp_ipc_handle(self.h, buf), "rc_tp_ipc_handle")
        return buf.raw

    def tp_open_peer(self, rank, handle):
        self._ck(self.L.rc_tp_open_peer(self.h, rank, C.c_char_p(handle)), "rc_tp_open_peer")

    def protect(self, ids, on):
        ids, on = _u64(ids), _u32(on)
        return self.L.rc_protect(self.h, ids.size, _p(ids), _p(on))

    def make_room(self, request_id, need, cap=4096):
        """Returns (status, ids): OK -> the claims demoted to make room; PROTECTED_CONFLICT -> blocking_claim_ids."""
        st, n = C.c_int32(-1), C.c_uint32()
        ids = np.zeros(cap, np.uint64)
        self._ck(self.L.rc_make_room(self.h, C.c_uint64(request_id), C.c_uint32(need), C.byref(st), _p(ids), cap,
                                     C.byref(n)), "rc_make_room")
        return st.value, [int(x) for x in ids[: min(cap, n.value)]]

    def protected_map(self):
        prot = np.zeros(self.NB, np.uint8)
        self._ck(self.L.rc_protected_map(self.h, _p(prot)), "rc_protected_map")
        return prot

    def wait(self, which):
        """Completes the oldest _begin of this kind and returns its status array.  A _begin that served nothing opened no
        operation in the library: its statuses were final at once and its wait() does not touch the library."""
        q = self._pending.get(which)
        if q and not q[0][2]:
            return q.pop(0)[1]
        self._ck(self.L.rc_wait(self.h, which), "rc_wait")
        return q.pop(0)[1] if q else None

    def test(self, which):
        """True if rc_wait(which) would not wait for a transfer."""
        d = C.c_int(0)
        self._ck(self.L.rc_test(self.h, which, C.byref(d)), "rc_test")
        return bool(d.value)

    def outcomes(self, cap=1 << 20):
        buf = np.zeros(cap, EVENT_DTYPE)
        n = C.c_uint64()
        self._ck(self.L.rc_outcomes(self.h, _p(buf), C.c_uint64(cap), C.byref(n)), "rc_outcomes")
        return buf[: n.value].copy()

    def set_faults(self, faults, flags=0):
        f = np.zeros(len(faults), FAULT_DTYPE)
        for i, (cid, kind, param) in enumerate(faults):
            f[i] = (cid, kind, param)
        return self.L.rc_set_faults(self.h, f.size, _p(f), flags)

    def claim_info(self, cid):
        o = ClaimInfo()
        if self.L.rc_claim_info(self.h, C.c_uint64(cid), C.byref(o)) != 0:
            return None
        return {k: getattr(o, k) for k, _ in ClaimInfo._fields_}

    def claim_blocks(self, cid):
        n = C.c_uint32()
        if self.L.rc_claim_blocks(self.h, C.c_uint64(cid), None, 0, C.byref(n)) != 0:
            return None
        buf = np.zeros(max(1, n.value), np.uint32)
        self._ck(self.L.rc_claim_blocks(self.h, C.c_uint64(cid), _p(buf), buf.size, C.byref(n)), "rc_claim_blocks")
        return buf[: n.value].copy()

    def claim_digests(self, cid, both=False):
        n = C.c_uint32()
        if self.L.rc_claim_digests(self.h, C.c_uint64(cid), None, None, 0, C.byref(n)) != 0:
            return None
        buf, buf2 = np.zeros(max(1, n.value), np.uint64), np.zeros(max(1, n.value), np.uint64)
        self._ck(self.L.rc_claim_digests(self.h, C.c_uint64(cid), _p(buf), _p(buf2), buf.size, C.byref(n)), "rc_claim_digests")
        return (buf[: n.value].copy(), buf2[: n.value].copy()) if both else buf[: n.value].copy()

    def host_read(self, cid):
        nbytes = C.c_uint64()
        if self.L.rc_host_read(self.h, C.c_uint64(cid), None, C.c_uint64(0), C.byref(nbytes)) != 0:
            return None
        out = np.zeros(nbytes.value, np.uint8)
        self.L.rc_host_read(self.h, C.c_uint64(cid), _p(out), C.c_uint64(out.size), C.byref(nbytes))
        return out

    def host_store(self, cid, block=0, n_blocks=1):
        """Borrowed read-only numpy view (no copy) of `n_blocks` host blocks of the claim starting at `block`;
        None if they are not contiguous in the pinned store or the claim holds no host bytes."""
        p, nbytes = C.c_void_p(), C.c_uint64()
        if self.L.rc_host_store(self.h, C.c_uint64(cid), block, C.byref(p), C.byref(nbytes)) != 0:
            return None
        if nbytes.value < n_blocks * self.blk:
            return None
        buf = (C.c_uint8 * (n_blocks * self.blk)).from_address(p.value)
        a = np.frombuffer(buf, np.uint8)
        a.flags.writeable = False
        return a

    def sync(self):
        self._ck(self.L.rc_sync(self.h), "rc_sync")
        for which in (0, 1):
            self._pending.pop(which, None)

    def pool_state(self):
        used = np.zeros(self.NB, np.uint8)
        ref = np.zeros(self.NB, np.uint32)
        self._ck(self.L.rc_pool_state(self.h, _p(used), _p(ref)), "rc_pool_state")
        return used, ref

    def stats(self):
        o = Stats()
        self._ck(self.L.rc_stats_get(self.h, C.byref(o)), "rc_stats_get")
        return {k: getattr(o, k) for k, _ in Stats._fields_}

    def stats_reset(self):
        self._ck(self.L.rc_stats_reset(self.h), "rc_stats_reset")

    def measure_link(self, nbytes, direction, reps=5):
        g = C.c_double()
        self._ck(self.L.rc_measure_link(self.h, C.c_uint64(nbytes), direction, reps, C.byref(g)), "rc_measure_link")
        return g.value

    def digest_blocks(self, src_ptr, n_blocks, want=True, both=False):
        d, e = np.zeros(n_blocks, np.uint64), np.zeros(n_blocks, np.uint64)
        ms = C.c_float()
        self._ck(self.L.rc_digest_blocks(self.h, C.c_void_p(src_ptr), n_blocks, _p(d) if want else None,
                                         _p(e) if want else None, C.byref(ms)), "rc_digest_blocks")
        return ((d, e) if both else d), ms.value


ERR_TOO_LARGE = -6
NOALLOC_MAX_PAGES = 32768


def digest_blocks_noalloc(src_ptr, n_blocks, layers, page_bytes, d_out_ptr, e_out_ptr, stream_ptr=0):
    """rc_digest_blocks_noalloc: device pointers in, nothing allocated, enqueued on the given stream.  Returns the code."""
    return lib().rc_digest_blocks_noalloc(C.c_void_p(src_ptr), C.c_uint32(n_blocks), C.c_uint32(layers), C.c_uint64(page_bytes),
                                          C.c_void_p(d_out_ptr), C.c_void_p(e_out_ptr), C.c_void_p(stream_ptr))


def validate_trace(events, want_claims=True):
    """rc_validate_trace over a numpy record array (EVENT_DTYPE).  Returns (report dict, per-claim records)."""
    ev = np.ascontiguousarray(events, dtype=EVENT_DTYPE)
    rep = TraceReport()
    cap = ev.size if want_claims else 0
    claims = np.zeros(max(1, cap), TRACE_CLAIM_DTYPE)
    rc = lib().rc_validate_trace(_p(ev), C.c_uint64(ev.size), C.byref(rep), _p(claims) if want_claims else None, C.c_uint64(cap))
    if rc != 0:
        raise RcError(rc, "rc_validate_trace")
    out = {k: getattr(rep, k) for k, _ in TraceReport._fields_ if k != "pad"}
    return out, claims[: min(cap, rep.n_claims)].copy()
