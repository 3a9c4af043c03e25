"""Build the CPU oracle (test infrastructure) into oracle/libbcf_oracle.so with gcc.

Usage: python oracle/build.py        (also called by __graft_entry__.build()).
Compiling the checker is not using it: nothing in the product path links or loads it.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "bcf_oracle.c")
HDR = os.path.join(HERE, "bcf_oracle_impl.h")
OUT = os.path.join(HERE, "libbcf_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(OUT):
        newest = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
        if os.path.getmtime(OUT) >= newest:
            return OUT
    cmd = ["gcc", "-O2", "-std=c11", "-Wall", "-Wextra", "-fPIC", "-shared", "-o", OUT, SRC]
    subprocess.check_call(cmd, cwd=HERE)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
