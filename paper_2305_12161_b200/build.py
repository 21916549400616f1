"""Build libising3d.so (C-ABI library, hand-written sm_100a kernels) in-tree with nvcc."""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libising3d.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    "-Xptxas", "-v",
    "-lcufft", "-Xlinker", "-rpath=/usr/local/cuda/lib64",
]


def sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC))


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = sources()
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(s) for s in srcs)):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = ["nvcc"] + NVCC_FLAGS + ["-o", tmp, os.path.join(CSRC, "ising3d.cu")]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building libising3d.so")
    if verbose:
        sys.stderr.write(res.stdout + res.stderr)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
