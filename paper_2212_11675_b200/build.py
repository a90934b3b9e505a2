"""Build libgsr_b200.so in-tree with nvcc for sm_100a (no JIT cache, no torch extension)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libgsr_b200.so")
SOURCES = ["gsr_matrix.cu", "gsr_aprod.cu", "gsr_lsqr.cu", "gsr_comm.cu", "gsr_constraints.cu",
           "gsr_static.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-ldl"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(_ROOT, "include", "gsr.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, extra_flags=(), out: str | None = None) -> str:
    """Build the library.  `extra_flags` (e.g. ["-DGSR_BOUNDS_CHECK"]: device asserts on the index
    computations of the product kernels) and `out` give a second, instrumented library beside
    the product one; binding.py loads it when GSR_B200_LIB names it (tests/test_gpu_bounds.py)."""
    target = out or LIB
    if force or out is not None or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = target + f".tmp{os.getpid()}"
        cmd = [nvcc, *NVCC_FLAGS, *extra_flags, "-I", os.path.join(_ROOT, "include"), "-I", CSRC, "-o", tmp,
               *[os.path.join(CSRC, s) for s in SOURCES]]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
            print(" ".join(cmd))
        subprocess.check_call(cmd)
        os.replace(tmp, target)
    return target


if __name__ == "__main__":
    print(build(force=True, verbose=True))
