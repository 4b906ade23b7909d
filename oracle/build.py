"""Builds oracle/libckf_oracle.so from oracle/ckf_oracle.cpp with g++ (no CUDA, no shared code).

-ffp-contract=off keeps the oracle the fixed point of the arithmetic (no FMA contraction), see
SURVEY.md §7 hard part 3.  Called by __graft_entry__.build() and lazily by oracle/__init__.py.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ckf_oracle.cpp")
LIB = os.path.join(HERE, "libckf_oracle.so")
FLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fPIC", "-shared", "-pthread", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.run(["g++", *FLAGS, SRC, "-o", tmp], check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
