"""Build oracle/libgray_oracle.so (TEST INFRASTRUCTURE, not product code).

    python oracle/build.py

Plain g++ -O2, no fast-math, no -march flags: the oracle is never tuned.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gray_oracle.cpp")
HDR = os.path.join(HERE, "gray_oracle.hpp")
LIB = os.path.join(HERE, "libgray_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB):
        newest = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
        if os.path.getmtime(LIB) >= newest:
            return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-pthread", "-ffp-contract=off",
           "-o", LIB, SRC]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
