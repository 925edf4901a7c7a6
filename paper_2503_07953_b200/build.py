"""Builds paper_2503_07953_b200/libmfc_b200.so (the C-ABI library of include/mfc_b200.h) with nvcc for sm_100a.

In-tree build: the .so sits next to this file, is git-ignored, and travels to the GPU box with the
snapshot.  nvcc cross-compiles without a GPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libmfc_b200.so")
SRC = [os.path.join(HERE, "csrc", "mfc_b200.cu")]
DEPS = SRC + [os.path.join(HERE, "csrc", "mfc_device.cuh"), os.path.join(ROOT, "include", "mfc_b200.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "--fmad=true", "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def _fresh() -> bool:
    return os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and _fresh():
        return LIB
    # several ranks of one job may get here together: one compiles (into a temporary, renamed when complete), the
    # others wait on the lock and find the library fresh
    import fcntl
    with open(LIB + ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if force or not _fresh():
                tmp = LIB + ".tmp.%d" % os.getpid()
                cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SRC
                subprocess.check_call(cmd)
                os.replace(tmp, LIB)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
