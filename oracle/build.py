"""Builds oracle/liboracle.so from oracle/cosmo_oracle.c with gcc.  TEST INFRASTRUCTURE (see the header of cosmo_oracle.c).

Plain `gcc -O2 -fopenmp`, no -ffast-math (long-double arithmetic must stay as written).
Called by __graft_entry__.build() and, on first use, by oracle/__init__.py (tests, smoke(), bench.py's oracle legs).
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "cosmo_oracle.c")
HDR = os.path.join(HERE, "gk21_nodes.h")
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(HDR))):
        return LIB
    cmd = ["gcc", "-std=gnu11", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-fno-fast-math", "-ffp-contract=off", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
