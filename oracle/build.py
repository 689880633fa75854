"""Build the CPU oracle (oracle/agnvar_oracle.cpp -> oracle/liboracle.so) with g++.

TEST INFRASTRUCTURE, NOT THE PRODUCT.  No CUDA, no code shared with paper_1909_06374_b200/csrc.
Usage:  python oracle/build.py          (also called by __graft_entry__.build() and tests/conftest.py)
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "agnvar_oracle.cpp")
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    # -ffp-contract=off: one rounding per written operation on any host (no effect on baseline x86-64, which has no FMA)
    cmd = ["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
