"""Compile the CPU oracle (oracle/oracle.cpp) into oracle/liboracle.so with g++.

TEST INFRASTRUCTURE. Building the checker is not using it: `__graft_entry__.build()` calls this;
only tests/, `__graft_entry__.smoke()` and bench.py's cpu_baseline / --impl reference legs load the result.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "oracle.cpp")
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    # -O2, no -ffast-math, no -march=native: plain IEEE double / x87 long double, portable to the GPU box's host.
    cmd = ["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-pthread", "-fno-fast-math", "-ffp-contract=off",
           SRC, "-o", LIB + ".tmp"]
    subprocess.check_call(cmd)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
