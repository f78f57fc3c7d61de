"""Build the CPU oracle (TEST INFRASTRUCTURE, not the product): g++ -> oracle/libu1gf_oracle.so.

`-ffp-contract=off` keeps every multiply and add separately rounded, so the oracle's arithmetic is
exactly what the source spells out.  Run as `python -m oracle.build` or via __graft_entry__.build().
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "u1gf_oracle.cpp")
LIB = os.path.join(HERE, "libu1gf_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
