"""Build step: compile the CUDA C-ABI library in-tree for sm_100a.

    python -m paper_2211_03193_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so stays beside the sources (git-ignored) so it travels
with the tree to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(CSRC, "libamh_b200.so")
SOURCES = ["amh_api.cu"]
PTXAS_LOG = os.path.join(CSRC, "ptxas_info.txt")        # registers / spills of the last build (git-ignored)


def deps():
    """Every file the library is built from: all of csrc/*.cu, csrc/*.cuh and the public header."""
    import glob
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh"))) + \
        [os.path.join(HERE, "..", "include", "amh.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "--fmad=true",            # no --use_fast_math: sqrtf/sincos/log stay IEEE-accurate
    "-Xcompiler", "-fPIC", "-shared",
    "-Xptxas", "-v",
]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in deps())


LIB_CHECKED = os.path.join(CSRC, "libamh_b200_checked.so")


def build_checked(force: bool = False) -> str:
    """The same library with -DAMH_CHECK: device-side range checks on every table / ring / shared-memory index of the
    pair loops (amh_check_status reports a failure).  For tests; the product path loads LIB."""
    if force or not os.path.exists(LIB_CHECKED) or any(os.path.getmtime(d) > os.path.getmtime(LIB_CHECKED) for d in deps()):
        tmp = LIB_CHECKED + ".tmp%d" % os.getpid()
        cmd = [nvcc()] + [f for f in NVCC_FLAGS if f not in ("-Xptxas", "-v")] + ["-DAMH_CHECK", "-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
        os.replace(tmp, LIB_CHECKED)
    return LIB_CHECKED


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        tmp = LIB + ".tmp%d" % os.getpid()
        cmd = [nvcc()] + NVCC_FLAGS + ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
        if verbose:
            sys.stderr.write(r.stderr)
        with open(PTXAS_LOG, "w") as f:
            f.write("# " + " ".join(cmd) + "\n" + r.stderr)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    if "--checked" in sys.argv:
        print(build_checked(force="--force" in sys.argv))
    else:
        print(build(force="--force" in sys.argv, verbose=True))
