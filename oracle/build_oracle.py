"""Compile the CPU oracle (oracle/xy_oracle.c) into oracle/liboracle.so with gcc.

TEST INFRASTRUCTURE, not the product.  Called by __graft_entry__.build() and, lazily, by
oracle/oracle.py.  -O2, no fast-math, no FMA contraction: the oracle's fp32 proposal
arithmetic (R5) must round exactly as written.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "xy_oracle.c")
LIB = os.path.join(HERE, "liboracle.so")

CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-fno-fast-math", "-ffp-contract=off",
          "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    hdr = os.path.join(HERE, "xy_oracle.h")
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(hdr))):
        return LIB
    cmd = ["gcc", *CFLAGS, SRC, "-o", LIB, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
