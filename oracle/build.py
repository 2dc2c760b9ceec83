"""Compile the fp64 CPU oracle (TEST INFRASTRUCTURE ONLY) into oracle/liboracle_ba.so with gcc."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCE = os.path.join(HERE, "oracle_ba.c")
HEADER = os.path.join(HERE, "oracle_ba.h")
LIBRARY = os.path.join(HERE, "liboracle_ba.so")


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(SOURCE), os.path.getmtime(HEADER))
    if not force and os.path.exists(LIBRARY) and os.path.getmtime(LIBRARY) >= newest:
        return LIBRARY
    # -ffp-contract=off: no fused multiply-adds, so the arithmetic is exactly the C source's.
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-Wall", "-Wextra",
           "-o", LIBRARY, SOURCE, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIBRARY


if __name__ == "__main__":
    print(build(force=True))
