"""Build libch.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1911_03386_b200.build [--force]
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libch.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17", "--fmad=true",
    "-Xcompiler", "-fPIC,-O2,-Wall", "--shared", "-cudart", "static",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cpp")))


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) \
        + [os.path.join(os.path.dirname(HERE), "include", "ch.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + sources()
        subprocess.run(cmd, check=True)
    return LIB


LIB_DEBUGSYNC = os.path.join(HERE, "libch_debugsync.so")


def build_debug_sync(force: bool = False) -> str:
    """libch_debugsync.so: the same library with -DCH_DEBUG_SYNC, i.e. with the in-kernel assertions on the sequence numbers
    of the flag-synchronised kernels (ch_line2d.cuh).  Load it with CH_LIBCH=<path> (binding.py)."""
    deps = sources() + glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh"))
    if force or not os.path.exists(LIB_DEBUGSYNC) or any(os.path.getmtime(d) > os.path.getmtime(LIB_DEBUGSYNC) for d in deps):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        subprocess.run([nvcc] + NVCC_FLAGS + ["-DCH_DEBUG_SYNC", "-o", LIB_DEBUGSYNC] + sources(), check=True)
    return LIB_DEBUGSYNC


if __name__ == "__main__":
    if "--debug-sync" in sys.argv:
        print(build_debug_sync(force="--force" in sys.argv))
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
