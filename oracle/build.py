"""Compile the CPU oracle (oracle/spin_oracle.c) into oracle/liboracle.so with gcc.

TEST INFRASTRUCTURE: the oracle is the checker, not the product.  Building it is not using it;
only tests/, bench.py's cpu_baseline / --impl reference legs and __graft_entry__.smoke() load it.
Flags: -O2, no FMA contraction, no -march (plain x86-64 SSE2 fp64, so results do not depend on the host CPU).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "spin_oracle.c")
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
           "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
