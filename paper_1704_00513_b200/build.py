"""Builds csrc/*.cu into paper_1704_00513_b200/libbfsc.so for sm_100a (in-tree, so the .so
travels to the GPU box with the repo snapshot). `python -m paper_1704_00513_b200.build`.
With BFSC_CHECKED=1 in the environment: libbfsc_checked.so, compiled with -DBFSC_CHECKED (every BFSC_CHECK of the kernels
counted instead of compiled away); binding.py loads that one under the same variable, and tests/conftest.py asserts at
the end of a run that no check failed: `BFSC_CHECKED=1 python -m pytest tests -m gpu`."""
from __future__ import annotations

import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
CHECKED = os.environ.get("BFSC_CHECKED", "") == "1"      # the bounds-asserting build (csrc/common.cuh: BFSC_CHECK), a library of its own
SO = os.path.join(HERE, "libbfsc_checked.so" if CHECKED else "libbfsc.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-shared", "--use_fast_math", "-Xptxas", "-v"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def stale() -> bool:
    if not os.path.exists(SO):
        return True
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "bfsc.h")]
    return os.path.getmtime(SO) < max(os.path.getmtime(p) for p in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        cmd = [NVCC] + FLAGS + (["-DBFSC_CHECKED"] if CHECKED else []) + ["-o", SO] + sources()
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode:
            print(r.stdout + r.stderr)
        if r.returncode:
            raise RuntimeError("nvcc failed")
    return SO


if __name__ == "__main__":
    build(force=True, verbose=True)
