"""Compile the oracle's C into oracle/libufnvc_oracle_f64.so and _f32.so (gcc, OpenMP).

Building the checker is not using it: __graft_entry__.build() calls this; the product never does.
x86-64-v3 (AVX2+FMA) rather than -march=native: the library is built on one box and run on another.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ufnvc_oracle.c")


def lib_path(real: str) -> str:
    return os.path.join(HERE, f"libufnvc_oracle_{real}.so")


def build(force: bool = False) -> None:
    for real, ctype in (("f64", "double"), ("f32", "float")):
        out = lib_path(real)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(SRC):
            continue
        cmd = ["gcc", "-O3", "-march=x86-64-v3", "-fopenmp", "-shared", "-fPIC",
               f"-DREAL={ctype}", SRC, "-o", out, "-lm"]
        subprocess.check_call(cmd)


if __name__ == "__main__":
    build(force="--force" in sys.argv)
