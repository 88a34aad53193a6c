"""Build the CPU oracle (test infrastructure) into oracle/libfestina_oracle.so.

g++ -O2 -ffp-contract=off: every fl(.) in the oracle must be one binary32 rounding, so FMA
contraction is disabled.  Called by __graft_entry__.build() and lazily by oracle/__init__.py.

FESTINA_ORACLE_SANITIZE=1 in the environment selects a second build of the same source with
-fsanitize=address,undefined (oracle/libfestina_oracle_san.so); tests/test_oracle_sanitizers.py runs the
pins against it in a child process with libasan preloaded.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "festina_oracle.cpp")
LIB = os.path.join(HERE, "libfestina_oracle.so")
LIB_SAN = os.path.join(HERE, "libfestina_oracle_san.so")
SAN_FLAGS = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined",
             "-fno-sanitize-recover=undefined"]


def sanitize() -> bool:
    return os.environ.get("FESTINA_ORACLE_SANITIZE", "0") == "1"


def build(force: bool = False) -> str:
    san = sanitize()
    lib = LIB_SAN if san else LIB
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= os.path.getmtime(SRC):
        return lib
    cmd = ["g++"] + (SAN_FLAGS if san else ["-O2"]) + ["-ffp-contract=off", "-std=c++17", "-shared", "-fPIC",
                                                        "-pthread", "-Wall", "-o", lib, SRC]
    subprocess.check_call(cmd)
    return lib


if __name__ == "__main__":
    print(build(force=True))
