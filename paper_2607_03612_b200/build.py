"""Build libsaf3r.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).  `python -m paper_2607_03612_b200.build`."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libsaf3r.so")
SOURCES = ["saf3r_api.cu"]
DEPS = ["saf3r_api.cu", "attn_kernel.cuh", "select_kernels.cuh", "token_kernels.cuh", "tokenwise_kernels.cuh", "ptx.cuh", os.path.join(ROOT, "include", "saf3r.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "--expt-relaxed-constexpr",
              "--expt-extended-lambda", "-Xcompiler", "-fPIC", "-shared", "-I", os.path.join(ROOT, "include")]


def nvcc_path() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.exists(p) or p == "nvcc"):
            return p
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    deps = [d if os.path.isabs(d) else os.path.join(CSRC, d) for d in DEPS]
    if not force and os.path.exists(OUT) and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in deps):
        return OUT
    cmd = [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", OUT] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd, cwd=CSRC)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
