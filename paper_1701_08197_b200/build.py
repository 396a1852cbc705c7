"""Builds the CUDA library in-tree: nvcc, sm_100a only, -lineinfo (no JIT cache, no torch extension).

    python -m paper_1701_08197_b200.build [--force]
"""
import os
import subprocess
import sys

_DIR = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_DIR, "csrc")
LIB = os.path.join(_DIR, "liblof.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-cudart", "static"]


def _sources():
    out = [os.path.join(_DIR, "..", "include", "lof.h")]
    for f in sorted(os.listdir(CSRC)):
        if f.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, f))
    return out


def build_lib(force=False, verbose=False):
    if os.environ.get("LOF_LIB_PATH"):
        return os.environ["LOF_LIB_PATH"]
    """Compile csrc/lof_api.cu (which includes every kernel header) into liblof.so."""
    srcs = _sources()
    if not force and os.path.exists(LIB) and all(os.path.getmtime(s) <= os.path.getmtime(LIB) for s in srcs):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("LOF_NVCC_EXTRA", "").split()      # e.g. -DLOF_FUSED_PROF for per-phase cycle counters
    cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", LIB, os.path.join(CSRC, "lof_api.cu")]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build_lib(force="--force" in sys.argv, verbose="-v" in sys.argv))
