"""Build libaton.so (hand-written CUDA for sm_100a) in-tree with nvcc.  No GPU is needed to compile."""
from __future__ import annotations

import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libaton.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-diag-suppress", "550",
              "--shared", "-Xcompiler", "-fPIC"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh"))
                  + [os.path.join(os.path.dirname(HERE), "include", "aton.h")])


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every csrc/*.cu (aton_api.cu holds the step kernels' instantiations) into libaton.so."""
    newest = max(os.path.getmtime(s) for s in sources())
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = LIB + f".{os.getpid()}.tmp"
    units = sorted(glob.glob(os.path.join(CSRC, "*.cu")))
    cmd = [nvcc] + NVCC_FLAGS + ["--threads", str(len(units))] + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", tmp] + units + ["-ldl"]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
