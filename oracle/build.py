"""Compile the CPU oracle (test infrastructure) into oracle/libkr_oracle.so with g++ -O2.

Run as ``python oracle/build.py``; ``__graft_entry__.build()`` calls ``build_oracle()`` too.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "kr_oracle.cpp")
LIB = os.path.join(HERE, "libkr_oracle.so")


def build_oracle(force: bool = False, verbose: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "kr_oracle.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-pthread", "-Wall", "-Wextra",
           "-o", LIB, SRC]
    if verbose:
        print(" ".join(cmd))
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build_oracle(force="--force" in sys.argv, verbose=True))
