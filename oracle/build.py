"""Build the CPU oracle (TEST INFRASTRUCTURE, not product) into oracle/libfarm_oracle.so with g++.

Flags matter: -ffp-contract=off and no fast-math so that rule R5's fp32 operations are rounded one by
one; -O2 as BASELINE.md states for the timed baseline.  Called by __graft_entry__.build(), tests/conftest.py
and bench.py's cpu_baseline / --impl reference legs.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "farm_oracle.cpp")
LIB = os.path.join(HERE, "libfarm_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-msse2", "-mfpmath=sse",
           "-shared", "-fPIC", "-o", LIB + ".tmp", SRC]
    subprocess.check_call(cmd)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
