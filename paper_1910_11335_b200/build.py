"""Build the CUDA library in-tree: nvcc -> paper_1910_11335_b200/libdoctors_b200.so (sm_100a only)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdoctors_b200.so")
SOURCES = ["api.cu", "host_tables.cpp"]
def _headers():
    """Every header the sources include: all of csrc/ plus the public header (a stale .so would be what the tests load)."""
    here = sorted(f for f in os.listdir(CSRC) if f.endswith((".cuh", ".h")))
    return here + [os.path.join("..", "..", "include", "doctors_b200.h")]


def _nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + _headers())


def build(force=False, verbose=False):
    """Compile every CUDA source for sm_100a into one shared library (no other arch, no fallback)."""
    if not force and not needs_build():
        return LIB
    cmd = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-shared", "-Xcompiler", "-fPIC",
           "-o", LIB] + [os.path.join(CSRC, f) for f in SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    cmd[1:1] = os.environ.get("DOCTORS_NVCC_FLAGS", "").split()
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
