"""ctypes wrapper over oracle/librc_oracle.so -- ORACLE, test infrastructure only.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this.  It imports nothing from the product package.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "librc_oracle.so")

EVENT_DTYPE = np.dtype([("seq", "<u8"), ("claim_id", "<u8"), ("code", "<u4"), ("aux", "<u4"), ("arg", "<u8")])
FAULT_DTYPE = np.dtype([("claim_id", "<u8"), ("kind", "<u4"), ("param", "<u4")])
TP_VERDICT_DTYPE = np.dtype([("flags", "<u4"), ("bad", "<u4")])      # flags: 1 served, 2 locally ok

EV_NAMES = {1: "ACCEPTED", 2: "MATERIALIZED", 3: "OFFLOADED", 4: "RESTORE_REQUIRED", 5: "LOAD_FAILED",
            6: "RESTORED", 7: "RESTORATION_FAILED", 8: "ACTIVE_REQUEST_REFUSED", 9: "DEMOTED", 10: "EXPIRED",
            11: "CONFLICT_REFUSED"}
REQ_FLAG = 0x80000000


class _Cfg(C.Structure):
    _fields_ = [("layers", C.c_uint32), ("kv_heads", C.c_uint32), ("head_dim", C.c_uint32),
                ("elem_bytes", C.c_uint32), ("block_size", C.c_uint32), ("pool_blocks", C.c_uint32),
                ("host_store_bytes", C.c_uint64), ("pool", C.c_void_p), ("fill", C.c_void_p)]


class _Info(C.Structure):
    _fields_ = [("claim_id", C.c_uint64), ("chain", C.c_uint64), ("host_bytes", C.c_uint64),
                ("state", C.c_uint32), ("P", C.c_uint32), ("N", C.c_uint32), ("M", C.c_uint32),
                ("nb", C.c_uint32), ("n_table", C.c_uint32)]


def build(force=False):
    src = os.path.join(_HERE, "rc_oracle.cpp")
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(src):
        subprocess.check_call(["sh", os.path.join(_HERE, "build.sh")])
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        for name in ("rco_mixL", "rco_mixF", "rco_mum", "rco_page_digest", "rco_block_digest", "rco_chain_of"):
            getattr(_lib, name).restype = C.c_uint64
        _lib.rco_mixL.argtypes = [C.c_uint64]
        _lib.rco_mixF.argtypes = [C.c_uint64]
        _lib.rco_mum.argtypes = [C.c_uint64, C.c_uint64]
        _lib.rco_page_digest.argtypes = [C.c_void_p, C.c_uint64, C.c_int]
        _lib.rco_block_digest.argtypes = [C.c_void_p, C.c_uint32, C.c_uint64, C.c_int]
        _lib.rco_chain_of.argtypes = [C.c_uint64, C.c_void_p, C.c_uint32]
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _u64(x):
    return np.ascontiguousarray(x, dtype=np.uint64)


def _u32(x):
    return np.ascontiguousarray(x, dtype=np.uint32)


def mixL(x):
    return int(lib().rco_mixL(C.c_uint64(x)))


def mixF(x):
    return int(lib().rco_mixF(C.c_uint64(x)))


def mum(x, y):
    return int(lib().rco_mum(C.c_uint64(x), C.c_uint64(y)))


def page_digest(page: np.ndarray, which=0):
    """which: 0 = the checksum family (d), 1 = the key-extension family (e)."""
    page = np.ascontiguousarray(page).view(np.uint8)
    return int(lib().rco_page_digest(_p(page), C.c_uint64(page.size), which))


def block_digest(blk: np.ndarray, n_pages: int, which=0):
    blk = np.ascontiguousarray(blk).view(np.uint8)
    return int(lib().rco_block_digest(_p(blk), n_pages, C.c_uint64(blk.size // n_pages), which))


def chain_of(claim_id, d):
    d = _u64(d)
    return int(lib().rco_chain_of(C.c_uint64(claim_id), _p(d), d.size))


class Oracle:
    """Oracle context over a HOST pool mirror (np.uint8, shape [L*2*NB*page]) and fill (np.uint8[NB]).

    Both arrays are borrowed and mutated in place by restore."""

    def __init__(self, layers, kv_heads, head_dim, elem_bytes, block_size, pool_blocks, pool, fill,
                 host_store_bytes=1 << 62):
        self.L = lib()
        page = block_size * kv_heads * head_dim * elem_bytes
        assert pool.dtype == np.uint8 and pool.flags.c_contiguous and pool.size == 2 * layers * pool_blocks * page
        assert fill.dtype == np.uint8 and fill.size == pool_blocks
        self.pool, self.fill = pool, fill
        self.page, self.blk, self.NB = page, 2 * layers * page, pool_blocks
        cfg = _Cfg(layers, kv_heads, head_dim, elem_bytes, block_size, pool_blocks, host_store_bytes,
                   pool.ctypes.data, fill.ctypes.data)
        self.h = C.c_void_p()
        rc = self.L.rco_create(C.byref(cfg), C.byref(self.h))
        if rc != 0:
            raise ValueError("rco_create failed: %d" % rc)

    def close(self):
        if self.h:
            self.L.rco_destroy(self.h)
            self.h = None

    def __del__(self):
        self.close()

    def mark_used(self, ids):
        ids = _u32(ids)
        return self.L.rco_mark_used(self.h, ids.size, _p(ids))

    def mark_free(self, ids):
        ids = _u32(ids)
        return self.L.rco_mark_free(self.h, ids.size, _p(ids))

    def accept(self, claim_ids, P, N, bt_off, bt_ids):
        claim_ids, P, N, bt_off, bt_ids = _u64(claim_ids), _u32(P), _u32(N), _u32(bt_off), _u32(bt_ids)
        st = np.zeros(claim_ids.size, np.int32)
        rc = self.L.rco_accept(self.h, claim_ids.size, _p(claim_ids), _p(P), _p(N), _p(bt_off), _p(bt_ids), _p(st))
        assert rc == 0
        return st

    def _batch(self, fn, claim_ids):
        claim_ids = _u64(claim_ids)
        st = np.zeros(claim_ids.size, np.int32)
        rc = fn(self.h, claim_ids.size, _p(claim_ids), _p(st))
        assert rc == 0
        return st

    def materialize(self, ids):
        return self._batch(self.L.rco_materialize, ids)

    def offload(self, ids):
        return self._batch(self.L.rco_offload, ids)

    def restore(self, ids):
        return self._batch(self.L.rco_restore, ids)

    def restore_request(self, request_id, ids):
        ids = _u64(ids)
        st = np.zeros(ids.size, np.int32)
        rc = self.L.rco_restore_request(self.h, C.c_uint64(request_id), ids.size, _p(ids), _p(st))
        assert rc == 0
        return st

    def set_policy(self, ids, policy):
        ids, policy = _u64(ids), _u32(policy)
        return self.L.rco_set_policy(self.h, ids.size, _p(ids), _p(policy))

    def release(self, ids):
        return self._batch(self.L.rco_release, ids)

    def set_tp(self, ranks):
        return self.L.rco_set_tp(self.h, ranks)

    def tp_restore_verify(self, ids):
        """Phase 1 of a TP-sharded restore: returns (statuses, local verdict records)."""
        ids = _u64(ids)
        st = np.zeros(ids.size, np.int32)
        v = np.zeros(ids.size, TP_VERDICT_DTYPE)
        rc = self.L.rco_tp_restore_verify(self.h, ids.size, _p(ids), _p(st), _p(v))
        if rc != 0:
            raise ValueError("rco_tp_restore_verify: %d" % rc)
        return st, v

    def tp_restore_commit(self, gathered, st):
        """Phase 2: gathered = verdict records of all ranks, shape [G, n]; completes the statuses of phase 1 in place."""
        g = np.ascontiguousarray(gathered, dtype=TP_VERDICT_DTYPE)
        rc = self.L.rco_tp_restore_commit(self.h, g.shape[1], g.shape[0], _p(g), _p(st))
        if rc != 0:
            raise ValueError("rco_tp_restore_commit: %d" % rc)
        return st

    def restore_begin(self, ids, request_id=0):
        """Split form (rc.h rc_restore_begin): phase 1 now; returns the statuses, -1 for served claims."""
        ids = _u64(ids)
        st = np.zeros(ids.size, np.int32)
        rc = self.L.rco_restore_begin(self.h, C.c_uint64(request_id), ids.size, _p(ids), _p(st))
        if rc != 0:
            raise ValueError("rco_restore_begin: %d" % rc)
        self._split_st = st
        return st

    def restore_end(self):
        """Split form (rc_wait(1)): phase 2; completes and returns the statuses of restore_begin."""
        rc = self.L.rco_restore_end(self.h, _p(self._split_st))
        if rc != 0:
            raise ValueError("rco_restore_end: %d" % rc)
        return self._split_st

    def protect(self, ids, on):
        ids, on = _u64(ids), _u32(on)
        return self.L.rco_protect(self.h, ids.size, _p(ids), _p(on))

    def make_room(self, request_id, need, cap=4096):
        """Returns (status, ids): OK -> the claims demoted to make room; PROTECTED_CONFLICT -> blocking_claim_ids."""
        st, n = C.c_int32(-1), C.c_uint32()
        ids = np.zeros(cap, np.uint64)
        rc = self.L.rco_make_room(self.h, C.c_uint64(request_id), C.c_uint32(need), C.byref(st), _p(ids), cap, C.byref(n))
        if rc != 0:
            raise ValueError("rco_make_room: %d" % rc)
        return st.value, [int(x) for x in ids[: min(cap, n.value)]]

    def protected_map(self):
        prot = np.zeros(self.NB, np.uint8)
        self.L.rco_protected_map(self.h, _p(prot))
        return prot

    def outcomes(self, cap=1 << 20):
        buf = np.zeros(cap, EVENT_DTYPE)
        n = C.c_uint64()
        self.L.rco_outcomes(self.h, _p(buf), C.c_uint64(cap), C.byref(n))
        return buf[: n.value].copy()

    def set_faults(self, faults, flags=0):
        f = np.zeros(len(faults), FAULT_DTYPE)
        for i, (cid, kind, param) in enumerate(faults):
            f[i] = (cid, kind, param)
        return self.L.rco_set_faults(self.h, f.size, _p(f), flags)

    def claim_info(self, cid):
        o = _Info()
        if self.L.rco_claim_info(self.h, C.c_uint64(cid), C.byref(o)) != 0:
            return None
        return {k: getattr(o, k) for k, _ in _Info._fields_}

    def claim_blocks(self, cid):
        n = C.c_uint32()
        buf = np.zeros(1 << 16, np.uint32)
        if self.L.rco_claim_blocks(self.h, C.c_uint64(cid), _p(buf), buf.size, C.byref(n)) != 0:
            return None
        if n.value > buf.size:
            buf = np.zeros(n.value, np.uint32)
            self.L.rco_claim_blocks(self.h, C.c_uint64(cid), _p(buf), buf.size, C.byref(n))
        return buf[: n.value].copy()

    def claim_digests(self, cid, both=False):
        """The claim's recorded per-block checksums d; both=True: (d, e) with e the key-extension digests."""
        n = C.c_uint32()
        buf, buf2 = np.zeros(1 << 16, np.uint64), np.zeros(1 << 16, np.uint64)
        if self.L.rco_claim_digests(self.h, C.c_uint64(cid), _p(buf), _p(buf2), buf.size, C.byref(n)) != 0:
            return None
        return (buf[: n.value].copy(), buf2[: n.value].copy()) if both else buf[: n.value].copy()

    def host_read(self, cid):
        nbytes = C.c_uint64()
        if self.L.rco_host_read(self.h, C.c_uint64(cid), None, C.c_uint64(0), C.byref(nbytes)) != 0:
            return None
        out = np.zeros(nbytes.value, np.uint8)
        self.L.rco_host_read(self.h, C.c_uint64(cid), _p(out), C.c_uint64(out.size), C.byref(nbytes))
        return out

    def pool_state(self):
        used = np.zeros(self.NB, np.uint8)
        ref = np.zeros(self.NB, np.uint32)
        self.L.rco_pool_state(self.h, _p(used), _p(ref))
        return used, ref

    def set_dedup(self, on=True):
        return self.L.rco_set_dedup(self.h, int(on))

    def set_layer_major(self, on=True):
        return self.L.rco_set_layer_major(self.h, int(on))

    def link_bytes(self):
        o = np.zeros(2, np.uint64)
        self.L.rco_link_bytes(self.h, _p(o))
        return int(o[0]), int(o[1])

    def stats(self):
        o = np.zeros(4, np.uint64)
        self.L.rco_stats(self.h, _p(o))
        return {"host_used": int(o[0]), "n_claims": int(o[1]), "n_events": int(o[2]), "generic_failures": int(o[3])}
