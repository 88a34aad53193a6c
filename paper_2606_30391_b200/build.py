"""Build libfestina_eval.so (the CUDA product library) in-tree with nvcc for sm_100a.

nvcc cross-compiles without a GPU.  -fmad=false is belt and braces: the kernels already use
__fmul_rn/__fadd_rn for every rounding the parity contract fixes.
"""
from __future__ import annotations

import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfestina_eval.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh"))
    deps.append(os.path.join(os.path.dirname(HERE), "include", "festina_eval.h"))
    return any(os.path.getmtime(p) > t for p in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    cmd = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-fmad=false", "-shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall",
           "-o", LIB] + sources()
    if verbose:
        cmd[1:1] = ["-Xptxas", "-v"]
    subprocess.check_call(cmd)
    return LIB


def sass_counts() -> str:
    """Per kernel of the built library: SASS size and how often the instructions that show the memory path
    (UBLKCP = 1-D TMA bulk copy, LDGSTS = cp.async, SYNCS = mbarrier, REDUX / CREDUX = warp reduction) and FFMA
    (none may appear where the parity contract fixes the rounding) occur: `python -m paper_2606_30391_b200.build --sass`."""
    import collections
    import re
    out = subprocess.run(["cuobjdump", "-sass", LIB], capture_output=True, text=True, check=True).stdout
    ops = ("UBLKCP", "LDGSTS", "SYNCS", "REDUX", "FFMA", "LDG", "LDS", "ATOM")
    rows, name, cnt, n = [], None, collections.Counter(), 0

    def flush():
        if name:
            rows.append((name, n, dict(cnt)))
    for line in out.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            flush()
            name, cnt, n = m.group(1), collections.Counter(), 0
            continue
        m = re.match(r"\s*/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
        if m and name:
            n += 1
            op = m.group(1)
            base = op.split(".")[0]
            base = {"CREDUX": "REDUX", "ATOMG": "ATOM", "ATOMS": "ATOM", "RED": "ATOM"}.get(base, base)
            if base in ops:
                cnt[base] += 1
    flush()
    demangle = subprocess.run(["c++filt"], input="\n".join(r[0] for r in rows), capture_output=True, text=True).stdout.splitlines()
    lines = ["| kernel | SASS instructions | " + " | ".join(ops) + " |", "|---|---|" + "---|" * len(ops)]
    for (nm, n, c), dn in sorted(zip(rows, demangle), key=lambda x: x[1]):
        short = re.sub(r"\(.*", "", dn.replace("(anonymous namespace)::", "").replace("<unnamed>::", "")).replace("void ", "")
        lines.append(f"| `{short}` | {n} | " + " | ".join(str(c.get(o, 0)) for o in ops) + " |")
    return "\n".join(lines)


if __name__ == "__main__":
    import sys
    if "--sass" in sys.argv:
        build()
        print(sass_counts())
    else:
        print(build(force=True, verbose="-v" in sys.argv))
