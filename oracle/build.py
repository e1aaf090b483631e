"""Build liboracle_sph.so from oracle/sph_oracle.c with gcc (test infrastructure; see sph_oracle.c header).

    python -m oracle.build

-ffp-contract=off: the neighbour predicate and the binary32 wrap are defined as fixed sequences of
individually rounded IEEE operations (readings R3/R4); the compiler must not fuse them.
"""
from __future__ import annotations
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sph_oracle.c")
LIB = os.path.join(HERE, "liboracle_sph.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
           "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
