"""Compile the C oracle into oracle/libmesh_ft_oracle.so (gcc -O2 -fopenmp, no fast-math).

Building the checker is not using it: __graft_entry__.build() calls this; only tests/, smoke() and
bench.py's cpu_baseline / --impl reference legs load the result.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mesh_ft_oracle.c")
LIB = os.path.join(HERE, "libmesh_ft_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-std=c11", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
