"""Build libsstepcg.so (the C-ABI library of include/sstep_cg.h) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsstepcg.so")
SOURCES = ["sstep_cg.cu"]
HEADERS = sorted(f for f in os.listdir(CSRC) if f.endswith(".cuh"))


def _newest_source_mtime() -> float:
    files = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(ROOT, "include", "sstep_cg.h")]
    return max(os.path.getmtime(f) for f in files)


def nvcc_command(out: str = LIB) -> list[str]:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    return [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
            "-I", os.path.join(ROOT, "include"), "--shared", "-Xcompiler", "-fPIC", "-o", out,
            *[os.path.join(CSRC, f) for f in SOURCES]]


def build_library(force: bool = False, verbose: bool = False) -> str:
    """Compile if the library is missing or older than its sources; returns its path."""
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < _newest_source_mtime():
        cmd = nvcc_command()
        if verbose:
            cmd[1:1] = ["-Xptxas", "-v"]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build_library(force=True, verbose=True))
