"""Build the CPU oracle shared library (test infrastructure; see oracle/gfcc_oracle.cpp header).

Usage:  python oracle/build.py     -> oracle/libgfcc_oracle.so  (g++ -O2 -fopenmp)
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gfcc_oracle.cpp")
LIB = os.path.join(HERE, "libgfcc_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", LIB, SRC]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
