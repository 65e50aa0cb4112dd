"""Compile the CPU oracle (oracle/pespace_oracle.cpp) into oracle/libpespace_oracle.so.

TEST INFRASTRUCTURE.  Building the checker is not using it: __graft_entry__.build()
calls this; only tests/, smoke() and bench.py's cpu_baseline / --impl reference legs load
the result.  Flags follow SURVEY.md section 7: no fast-math, no FMA contraction.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "pespace_oracle.cpp")
HDR = os.path.join(HERE, "pespace_oracle.h")
LIB = os.path.join(HERE, "libpespace_oracle.so")

FLAGS = ["-O2", "-std=gnu++17", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
         "-shared", "-fPIC", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    stale = (not os.path.exists(LIB)
             or os.path.getmtime(LIB) < max(os.path.getmtime(SRC), os.path.getmtime(HDR)))
    if force or stale:
        cmd = ["g++", *FLAGS, SRC, "-o", LIB, "-lquadmath", "-lm"]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
