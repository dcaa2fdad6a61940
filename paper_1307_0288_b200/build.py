"""In-tree build of libkg.so (CUDA, sm_100a) with nvcc.  `python -m paper_1307_0288_b200.build`."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SRC = [os.path.join(HERE, "csrc", "kg.cu")]
DEPS = SRC + [os.path.join(HERE, "csrc", "kg_kernels.cuh"), os.path.join(HERE, "csrc", "kg_staged.cuh"), os.path.join(ROOT, "include", "kg.h")]
LIB = os.path.join(HERE, "libkg.so")

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def build(force: bool = False, verbose: bool = False) -> str:
    newest = max(os.path.getmtime(p) for p in DEPS)
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < newest:
        nvcc = os.environ.get("NVCC", "nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-I", os.path.join(ROOT, "include"), "-o", LIB] + SRC
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
