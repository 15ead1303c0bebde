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
