"""Builds libclt.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1812_00525_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with gpurun.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libclt.so")
# the same library with the textbook RK4 accumulator schedule (-DCLT_TEXTBOOK_RK4): the A/B that measures what the
# reduced-traffic schedule costs in round-off (tests/test_parity_gpu.py); never the default
LIB_TEXTBOOK = os.path.join(HERE, "libclt_textbook.so")
SOURCES = ["clt_api.cu", "clt_kernels.cu"]
HEADERS = [os.path.join(CSRC, "clt_internal.h"), os.path.join(ROOT, "include", "clt.h")]

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall", "-shared", "-Xptxas", "-v",
    "-Xfatbin", "-compress-all",      # the -lineinfo sections (PTX text, line tables) are 80 % of the cubin
]


def _stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(lib: str, defines, logname: str, verbose: bool) -> None:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = lib + f".tmp{os.getpid()}"
    cmd = [nvcc] + NVCC_FLAGS + list(defines) + ["-I", os.path.join(ROOT, "include"), "-I", CSRC, "-o", tmp] + \
          [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = res.stdout + res.stderr
    with open(os.path.join(HERE, logname), "w") as f:
        f.write(" ".join(cmd) + "\n" + log)
    if res.returncode != 0:
        sys.stderr.write(log)
        raise RuntimeError(f"nvcc failed building {os.path.basename(lib)}")
    if verbose:
        print(log)
    os.replace(tmp, lib)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale(LIB):
        _compile(LIB, [], "build.log", verbose)
    return LIB


def build_textbook(force: bool = False, verbose: bool = False) -> str:
    """libclt_textbook.so: same sources, textbook RK4 accumulator schedule (A/B for the parity tests only)."""
    if force or _stale(LIB_TEXTBOOK):
        _compile(LIB_TEXTBOOK, ["-DCLT_TEXTBOOK_RK4"], "build_textbook.log", verbose)
    return LIB_TEXTBOOK


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
    if "--textbook" in sys.argv:
        print(build_textbook(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
