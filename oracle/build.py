"""Compile oracle/cbct_oracle.c and oracle/siddon_oracle.c into oracle/libcbct_oracle.so with gcc (fp64, OpenMP).

Building the checker is not using it: __graft_entry__.build() calls this, the product
path never loads the result.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRCS = [os.path.join(HERE, "cbct_oracle.c"), os.path.join(HERE, "siddon_oracle.c")]
LIB = os.path.join(HERE, "libcbct_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(s) for s in SRCS):
        return LIB
    # -O2 without -ffast-math: keep IEEE fp64 semantics; -ffp-contract=off: no fused multiply-adds
    cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-Wall", "-Wextra", "-o", LIB + ".tmp", *SRCS, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
