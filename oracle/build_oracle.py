"""Compile oracle/triples_oracle.c into oracle/liboracle_triples.so with gcc.

TEST INFRASTRUCTURE (see oracle/__init__.py).  Building the checker is not using it:
__graft_entry__.build() calls build() here.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "triples_oracle.c")
LIB = os.path.join(HERE, "liboracle_triples.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    # -O2, no -ffast-math: keep IEEE semantics; -fopenmp as in the paper's CPU code (L121).
    cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
