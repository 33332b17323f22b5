"""Build the CPU oracle (TEST INFRASTRUCTURE) into oracle/liborc_mps.so.

g++ -O2 -ffp-contract=off: no FMA contraction, no fast-math, so the distance
test r2 = (dx*dx + dy*dy) + dz*dz rounds exactly as DESIGN.md reading Q2 says.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mps_oracle.cpp")
LIB = os.path.join(HERE, "liborc_mps.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math",
           "-shared", "-fPIC", "-o", LIB, SRC]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
