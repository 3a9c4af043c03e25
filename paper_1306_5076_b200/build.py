"""Build libbcf.so (the C-ABI CUDA library, include/bcf.h) in-tree with nvcc for sm_100a.

Usage: python -m paper_1306_5076_b200.build [--force]      (also called by __graft_entry__.build()).
nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with gpurun.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libbcf.so")
SOURCES = ["bcf_api.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-shared", "-Xcompiler", "-fPIC",
]


def _newest_source_mtime():
    newest = os.path.getmtime(os.path.join(HERE, "..", "include", "bcf.h"))
    for f in os.listdir(CSRC):
        newest = max(newest, os.path.getmtime(os.path.join(CSRC, f)))
    return newest


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(OUT) and os.path.getmtime(OUT) >= _newest_source_mtime():
        return OUT
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", OUT] + \
        [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd, cwd=HERE)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
