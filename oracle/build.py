"""Build the CPU oracle shared library (test infrastructure).  `python -m oracle.build`."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "bte_oracle.cpp")
LIB = os.path.join(HERE, "libbte_oracle.so")

# -ffp-contract=off: no FMA contraction -- every operation rounds once, in the written order.
CMD = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", LIB, SRC]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    subprocess.run(CMD, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
