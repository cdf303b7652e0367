"""Build the CPU oracle shared library (test infrastructure; see ns_oracle.cpp header).

Usage: python oracle/build.py   ->  oracle/libns_oracle.so
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRCS = [os.path.join(HERE, "ns_oracle.cpp"), os.path.join(HERE, "ns2d_oracle.cpp")]   # 3-D and 2-D oracles, no shared code
LIB = os.path.join(HERE, "libns_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(f) for f in SRCS):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", *SRCS, "-o", LIB]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
