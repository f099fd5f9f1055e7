"""Build step of libgint.so (in-tree, sm_100a only): `python -m paper_2409_09399_b200.build`."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgint.so")
SOURCES = ("gint_init.cu", "gint_kernels.cu", "gint_force.cu")
NVCC_FLAGS = ("-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "gint.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/*.cu into paper_2409_09399_b200/libgint.so with nvcc (cross-compiles without a GPU)."""
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    extra = os.environ.get("GINT_NVCC_EXTRA", "").split()      # developer switches (e.g. -DGINT_DBG_NO_MMA); empty in normal builds
    cmd = [nvcc, *NVCC_FLAGS, *extra, *(("-Xptxas", "-v") if verbose else ()), "-o", LIB,
           *(os.path.join(CSRC, s) for s in SOURCES)]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
