"""Build the CPU oracle shared library (test infrastructure, see mq_oracle.cpp header).

    python oracle/build.py            # -> oracle/libmq_oracle.so

-O2 -ffp-contract=off: no FMA contraction, so the binary32 divisions of Eq.1 are the
literal IEEE operations.  The same flags are used when bench.py times the oracle
("the oracle as it stands").
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mq_oracle.cpp")
OUT = os.path.join(HERE, "libmq_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(OUT) and os.path.getmtime(OUT) >= os.path.getmtime(SRC):
        return OUT
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
           "-Wall", "-Wextra", "-o", OUT, SRC]
    subprocess.check_call(cmd)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
