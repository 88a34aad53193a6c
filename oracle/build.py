"""Build the CPU oracle (test infrastructure) into oracle/libfestina_oracle.so.

g++ -O2 -ffp-contract=off: every fl(.) in the oracle must be one binary32 rounding, so FMA
contraction is disabled.  Called by __graft_entry__.build() and lazily by oracle/__init__.py.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "festina_oracle.cpp")
LIB = os.path.join(HERE, "libfestina_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", "-pthread",
           "-Wall", "-o", LIB, SRC]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
