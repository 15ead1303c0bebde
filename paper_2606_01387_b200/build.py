"""Builds paper_2606_01387_b200/librc.so (sm_100a only) in-tree with nvcc.

`python -m paper_2606_01387_b200.build` or `build()`; rebuilds when a source is newer.
"""
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
SO = os.path.join(_HERE, "librc.so")
SRCS = [os.path.join(_HERE, "csrc", "librc.cu")]
DEPS = [os.path.join(_HERE, "csrc", f) for f in sorted(os.listdir(os.path.join(_HERE, "csrc")))] + [
    os.path.join(os.path.dirname(_HERE), "include", "rc.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-shared", "-cudart", "shared"]


def build(force=False, verbose=False):
    if not force and os.path.exists(SO) and all(os.path.getmtime(SO) >= os.path.getmtime(d) for d in DEPS):
        return SO
    cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", SO] + SRCS
    subprocess.check_call(cmd)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
