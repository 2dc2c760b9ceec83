"""Compile the CUDA library IN-TREE: paper_2605_30583_b200/libcaspar_ba.so (sm_100a only)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIBRARY = os.path.join(HERE, "libcaspar_ba.so")
SOURCES = ["ba_api.cu", "ba_kernels.cu", "ba_reorder.cpp"]
HEADERS = [os.path.join(CSRC, "ba_internal.h"), os.path.join(HERE, "..", "include", "caspar_ba.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC,-fopenmp,-O3", "-shared", "-lgomp"]


def is_stale() -> bool:
    if not os.path.exists(LIBRARY):
        return True
    built = os.path.getmtime(LIBRARY)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > built for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not is_stale():
        return LIBRARY
    cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIBRARY] + SOURCES
    subprocess.run(cmd, check=True, cwd=CSRC)
    return LIBRARY


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
