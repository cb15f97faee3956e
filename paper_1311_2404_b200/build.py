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
# one translation unit for the C ABI and one per <lattice, real> pair of kernel instantiations
SOURCES = [os.path.join(CSRC, n) for n in ("lbm_b200.cu", "lbm_impl_d2q9_f32.cu", "lbm_impl_d2q9_f64.cu",
                                           "lbm_impl_d3q19_f32.cu", "lbm_impl_d3q19_f64.cu")]
HEADERS = [os.path.join(CSRC, n) for n in ("lbm_impl.cuh", "lbm_kernels.cuh", "lbm_node.cuh", "lbm_lattice.cuh")] + [
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
        objs, procs = [], []
        for src in SOURCES:  # the translation units are independent: compile them side by side
            obj = os.path.join(OBJDIR, os.path.basename(src)[:-3] + ".o")
            objs.append(obj)
            procs.append((src, subprocess.Popen([nvcc()] + NVCC_FLAGS + extra + ["-c", "-o", obj, src])))
        failed = [src for src, p in procs if p.wait() != 0]
        if failed:
            raise RuntimeError("nvcc failed on " + ", ".join(failed))
        tmp = LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call([nvcc(), "-shared", "-o", tmp] + objs)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
