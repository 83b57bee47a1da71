"""Build the C-ABI shared library (libgpw.so) in-tree with nvcc for sm_100a.

    python -m paper_2603_24881_b200.build [--force]

The library holds the host plan builder (csrc/plan.cpp) and the CUDA kernels plus the C ABI
(csrc/gpw_api.cu, pairs_device.cu, plan_device.cu, pairpass.cu, collocate.cu, integrate.cu, interp.cu); include/gpw.h is the interface.  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgpw.so")
SOURCES = ["plan.cpp", "pairs_device.cu", "plan_device.cu", "gpw_api.cu", "pairpass.cu", "pairpass_reg_pre.cu", "pairpass_reg_post.cu", "collocate.cu", "integrate.cu", "interp.cu"]
HEADERS = ["gpw_internal.h", "gpw_math.cuh", "gpw_kernels.cuh", "pairpass.cuh", "pairpass_reg.cuh", "pairpass_reg_kernel.cuh", "plan_device.h"]
# plan_device.cu repeats the host builder's geometric block test: no FMA contraction, so that the two agree bit for bit
EXTRA = {"plan_device.cu": ["-fmad=false"], "pairs_device.cu": ["-fmad=false"]}
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-O3", "-I", os.path.join(ROOT, "include"), "-I", CSRC]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(ROOT, "include", "gpw.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    # one builder at a time (torchrun ranks start together): the others wait, then find the library fresh
    import fcntl
    with open(os.path.join(HERE, ".build.lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and not _stale():
                return LIB
            return _build_locked(verbose, force)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)


def _build_locked(verbose: bool, force: bool = False) -> str:
    """Compile what is out of date (an object is rebuilt when its source, any header or this file is newer), in
    parallel, then link."""
    hdrs = [os.path.join(CSRC, f) for f in HEADERS] + [os.path.join(ROOT, "include", "gpw.h"), os.path.abspath(__file__)]
    hdr_t = max(os.path.getmtime(h) for h in hdrs)
    objs = []
    procs = []
    for src in SOURCES:
        obj = os.path.join(CSRC, os.path.splitext(src)[0] + ".o")
        objs.append(obj)
        path = os.path.join(CSRC, src)
        if not force and os.path.exists(obj) and os.path.getmtime(obj) > max(hdr_t, os.path.getmtime(path)):
            continue
        cmd = [NVCC] + FLAGS + EXTRA.get(src, []) + (["-Xptxas", "-v"] if verbose else []) + ["-c", path, "-o", obj]
        procs.append((cmd, subprocess.Popen(cmd)))
    for cmd, p in procs:
        if p.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    cmd = [NVCC, "-shared", "-o", LIB] + objs + ["-lcufft"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
