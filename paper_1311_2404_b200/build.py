"""Build step: compile csrc/lbm_b200.cu into paper_1311_2404_b200/liblbm_b200.so for sm_100a.

nvcc cross-compiles without a GPU.  The library is built in-tree so that it travels with the
repository snapshot to the GPU box.  No --use_fast_math: FTZ and approximate division would
break parity with the oracle (the paper saw FTZ crash a model).
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "liblbm_b200.so")
OBJDIR = os.path.join(_HERE, "build")
# one translation unit for the C ABI, one per <lattice, real> pair for the conversion kernels, and
# one per <lattice, real, model> for the step kernels: they are independent and compile side by side
SOURCES = [os.path.join(CSRC, "lbm_b200.cu"), os.path.join(CSRC, "lbm_noalloc.cu")] + [
    os.path.join(CSRC, "lbm_impl_%s_%s.cu" % (lat, pr)) for lat in ("d2q9", "d3q19") for pr in ("f32", "f64")] + [
    os.path.join(CSRC, "lbm_step_%s_%s_%s.cu" % (lat, pr, m))
    for lat in ("d3q19", "d2q9") for pr in ("f32", "f64") for m in ("bgk", "mrt", "sc", "reg", "les")]
HEADERS = [os.path.join(CSRC, n) for n in ("lbm_impl.cuh", "lbm_steps.cuh", "lbm_kernels.cuh", "lbm_node.cuh", "lbm_lattice.cuh")] + [
    os.path.join(os.path.dirname(_HERE), "include", "lbm.h")]

NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC,-fvisibility=hidden"]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: cannot build liblbm_b200.so")
    return exe


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in SOURCES + HEADERS + [os.path.abspath(__file__)])


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile the library if it is missing or older than its sources; return its path."""
    if force or stale():
        os.makedirs(OBJDIR, exist_ok=True)
        extra = (["-Xptxas", "-v"] if verbose else []) + os.environ.get("LBM_NVCC_EXTRA", "").split()
        objs, jobs = [], []
        for src in SOURCES:
            obj = os.path.join(OBJDIR, os.path.basename(src)[:-3] + ".o")
            objs.append(obj)
            jobs.append((src, [nvcc()] + NVCC_FLAGS + extra + ["-c", "-o", obj, src]))
        failed, running, width = [], [], max(2, os.cpu_count() or 2)
        while jobs or running:  # at most one nvcc per core
            while jobs and len(running) < width:
                src, cmd = jobs.pop(0)
                running.append((src, subprocess.Popen(cmd)))
            src, proc = running.pop(0)
            if proc.wait() != 0:
                failed.append(src)
        if failed:
            raise RuntimeError("nvcc failed on " + ", ".join(failed))
        tmp = LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call([nvcc(), "-shared", "-o", tmp] + objs)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
