"""Compile oracle/das_oracle.c into oracle/libdas_oracle.so (TEST INFRASTRUCTURE).

gcc -O2, no fast-math, no FMA contraction, OpenMP over voxels.
Building the checker is not using it: __graft_entry__.build() may call this."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "das_oracle.c")
LIB = os.path.join(HERE, "libdas_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
           "-shared", "-fPIC", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
