"""Builds paper_2505_22822_b200/libckf.so in-tree with nvcc for sm_100a (no torch extension machinery needed:
the boundary is a plain C ABI)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libckf.so")
SOURCES = ["ckf.cu"]
DEPS = ["ckf.cu", "ckf_math.cuh", "ckf_nav.cuh", "ckf_kernels.cuh", "ckf_step.cuh", "ckf_fit.cuh", "ckf_visit.cuh", "ckf_branch.cuh", "ckf_emit.cuh", "ckf_sort.cuh", "ckf_peak.cuh", "ckf_resolve.cuh", "ckf_seed.cuh",
        "ckf_host_geom.h", os.path.join("..", "..", "include", "ckf.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def up_to_date() -> bool:
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(os.path.join(CSRC, d)) <= t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and up_to_date():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [nvcc, *NVCC_FLAGS, *[os.path.join(CSRC, s) for s in SOURCES], "-o", tmp]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    os.replace(tmp, LIB)
    with open(os.path.join(HERE, "ptxas_info.txt"), "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stderr)
    if verbose:
        print(r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
