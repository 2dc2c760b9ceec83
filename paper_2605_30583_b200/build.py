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


def ptxas_table() -> str:
    """Registers / stack / spills / static shared memory of every kernel, from `nvcc -Xptxas -v` (evidence for
    profiles/: `python -m paper_2605_30583_b200.build --ptxas-table`)."""
    import re
    import tempfile

    rows = []
    with tempfile.TemporaryDirectory() as tmp:
        cmd = [NVCC, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xptxas", "-v",
               "-c", "ba_kernels.cu", "-o", os.path.join(tmp, "k.o")]
        txt = subprocess.run(cmd, check=True, cwd=CSRC, capture_output=True, text=True).stderr
    pat = re.compile(r"Compiling entry function '([^']+)'.*?\n.*?\n\s+(\d+) bytes stack frame, (\d+) bytes spill stores, "
                     r"(\d+) bytes spill loads\n.*?Used (\d+) registers(?:, used (\d+) barriers)?(?:, (\d+) bytes smem)?")
    ents = pat.findall(txt)
    names = subprocess.run(["c++filt"] + [e[0] for e in ents], capture_output=True, text=True).stdout.splitlines()
    rows.append("| kernel | registers | stack B | spill stores / loads B | static smem B |")
    rows.append("|---|---|---|---|---|")
    for n, e in zip(names, ents):
        n = re.sub(r"\(.*", "", n.replace("cba::", "").replace("void ", ""))
        rows.append(f"| `{n}` | {e[4]} | {e[1]} | {e[2]} / {e[3]} | {e[6] or 0} |")
    return "\n".join(rows)


def sass_evidence() -> str:
    """The instructions that prove the TMA / mbarrier path in the built library's two persistent kernels
    (`python -m paper_2605_30583_b200.build --sass-evidence`): UBLKCP (cp.async.bulk), SYNCS (mbarrier),
    FENCE.VIEW.ASYNC (fence.proxy.async), RED / ATOM, with their counts and the first occurrence of each in context."""
    import collections
    import re

    build()
    names = subprocess.run(["cuobjdump", "-sass", LIBRARY], capture_output=True, text=True, check=True).stdout
    out = []
    for kernel in ("schur_matvec_pipelined_kernelILi256ELi3ELb0ELi0E", "linearize_pipelined_kernelILi256ELi3ELb1E"):
        m = re.search(r"Function : (\S*%s\S*)" % kernel, names)
        if not m:
            continue
        fn = m.group(1)
        sass = subprocess.run(["cuobjdump", "-sass", "-fun", fn, LIBRARY], capture_output=True, text=True).stdout
        lines = [re.sub(r"\s*/\* 0x[0-9a-f]+ \*/\s*$", "", ln) for ln in sass.splitlines() if re.search(r"/\*[0-9a-f]{4}\*/", ln)]
        demangled = subprocess.run(["c++filt", fn], capture_output=True, text=True).stdout.strip()
        out.append(f"## `{demangled}` ({len(lines)} SASS instructions)\n")
        counts = collections.Counter()
        first = {}
        pat = re.compile(r"\b(UBLKCP\S*|SYNCS\.\S+|FENCE\.VIEW\.ASYNC\S*|REDG?\.\S+|ATOM[SG]?\.\S+|BAR\.\S+|MEMBAR\.\S+)")
        for i, ln in enumerate(lines):
            mm = pat.search(ln)
            if mm:
                counts[mm.group(1)] += 1
                first.setdefault(mm.group(1), i)
        out.append("| mnemonic | count |\n|---|---|")
        out += [f"| `{k}` | {v} |" for k, v in sorted(counts.items())]
        out.append("\nFirst occurrence of each, with the two instructions before and after:\n\n```")
        for k, i in sorted(first.items(), key=lambda x: x[1]):
            out += [ln.strip() for ln in lines[max(0, i - 2):i + 3]] + ["..."]
        out.append("```\n")
    return "\n".join(out)


if __name__ == "__main__":
    import sys
    if "--sass-evidence" in sys.argv:
        print(sass_evidence())
    elif "--ptxas-table" in sys.argv:
        print(ptxas_table())
    else:
        print(build(force=True, verbose="-v" in sys.argv))
