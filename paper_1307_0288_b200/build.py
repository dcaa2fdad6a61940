"""In-tree build of libkg.so (CUDA, sm_100a) with nvcc.  `python -m paper_1307_0288_b200.build`.

The library is eight translation units — kg.cu (C ABI, drivers, one-thread-per-element kernels)
one kg_staged_k<K>.cu per compiled neighbour-list row width and kg_tb2.cu (two-step kernels) — compiled in parallel and linked
with the CUDA runtime statically (no libtorch)."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
SRC = [os.path.join(CSRC, f) for f in ("kg.cu", "kg_staged_k2.cu", "kg_staged_k3.cu", "kg_staged_k4.cu",
                                       "kg_staged_k6.cu", "kg_staged_k9.cu", "kg_tb2.cu", "kg_small.cu")]
HEADERS = [os.path.join(CSRC, f) for f in ("kg_common.cuh", "kg_kernels.cuh", "kg_staged.cuh",
                                           "kg_staged_impl.cuh", "kg_staged_launch.h", "kg_partition.h",
                                           "kg_tb2.cuh", "kg_tb2_launch.h", "kg_small.cuh", "kg_small_launch.h", "kg_smem_config.h")]
DEPS = SRC + HEADERS + [os.path.join(ROOT, "include", "kg.h")]
LIB = os.path.join(HERE, "libkg.so")
OBJ_DIR = os.path.join(HERE, "build")

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC"]


def build(force: bool = False, verbose: bool = False) -> str:
    newest = max(os.path.getmtime(p) for p in DEPS)
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < newest:
        nvcc = os.environ.get("NVCC", "nvcc")
        os.makedirs(OBJ_DIR, exist_ok=True)
        objs = [os.path.join(OBJ_DIR, os.path.basename(s)[:-3] + ".o") for s in SRC]

        def compile_one(pair):
            src, obj = pair
            cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
                  ["-I", os.path.join(ROOT, "include"), "-c", "-o", obj, src]
            return subprocess.run(cmd, check=True, capture_output=verbose, text=True)

        with ThreadPoolExecutor(max_workers=len(SRC)) as pool:
            for r in pool.map(compile_one, zip(SRC, objs)):
                if verbose:
                    sys.stderr.write(r.stderr)
        subprocess.run([nvcc, "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a",
                        "-o", LIB] + objs, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
