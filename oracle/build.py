"""Compile the C oracle (test infrastructure) into oracle/libmbscb_oracle.so.

    python -m oracle.build

-O2, no fast-math, OpenMP for the paper's CPU threading (threads over cells for
OCI, over angles for SI).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mbscb_oracle.c")
LIB = os.path.join(HERE, "libmbscb_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC", "-Wall", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
