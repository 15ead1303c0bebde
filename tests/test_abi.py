"""The C-ABI library loads and exports every symbol include/rc.h declares (no compute calls
without a GPU); the product path fails loudly when no CUDA device is present."""
import ctypes
import os
import re

import pytest

from paper_2606_01387_b200 import build as B, rc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "rc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(?:int|const char\*)\s+(rc_[a-z_]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    lib = ctypes.CDLL(B.build())
    names = _declared()
    assert len(names) >= 25
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(rc.EXPORTS) == names


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    cfg = rc.Config(2, 2, 64, 2, 16, 256, 64, 4096, 4096, 2, 1 << 20, 1 << 20, 256, 256, 0, 0, 0, 0, 0, 0, 0, 0, 0)
    h = ctypes.c_void_p()
    assert rc.lib().rc_create(ctypes.byref(cfg), ctypes.byref(h)) == rc.ERR_CUDA and not h.value


def test_rc_create_rejects_bad_geometry():
    h = ctypes.c_void_p()
    cfg = rc.Config(2, 2, 64, 2, 3, 256, 64, 4096, 4096, 2, 1 << 20, 1 << 20, 256, 256, 0, 0, 0, 0, 0, 0, 0, 0, 0)  # page % 4096 != 0
    assert rc.lib().rc_create(ctypes.byref(cfg), ctypes.byref(h)) == rc.ERR_INVALID
    assert rc.lib().rc_strerror(rc.ERR_CAPACITY).decode().startswith("capacity")


def test_noalloc_entry_point_validates_before_it_touches_the_device():
    L = rc.lib()
    big = rc.NOALLOC_MAX_PAGES // 4 + 1                        # layers = 2 -> 4 pages per block
    assert rc.digest_blocks_noalloc(256, big, 2, 4096, 256, 256) == rc.ERR_TOO_LARGE
    assert "scratch" in L.rc_strerror(rc.ERR_TOO_LARGE).decode()
    assert rc.digest_blocks_noalloc(256, 1, 2, 4096 + 64, 256, 256) == rc.ERR_INVALID       # page % 4096
    assert rc.digest_blocks_noalloc(264, 1, 2, 4096, 256, 256) == rc.ERR_INVALID            # source alignment
    assert rc.digest_blocks_noalloc(0, 0, 2, 4096, 0, 0) == 0                               # empty range
