"""Compile oracle/roadrunner_oracle.c into oracle/libroadrunner_oracle.so (gcc, -O2, scalar fp64).

TEST INFRASTRUCTURE.  Called by ``oracle.load()`` when the library is missing or older than its
source, and by ``__graft_entry__.build()`` (building the checker is not using it).
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "roadrunner_oracle.c")
LIB = os.path.join(HERE, "libroadrunner_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    # -ffp-contract=off: no FMA contraction, so the arithmetic is the formula as written
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-Wall", "-Wextra", "-o", tmp, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
