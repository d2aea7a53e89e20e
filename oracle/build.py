"""Build the CPU oracle (test infrastructure) into oracle/libref_lbm.so.

    python oracle/build.py

-ffp-contract=off: no FMA contraction, so every operation in ref_lbm.cpp is one
IEEE-754 rounding.  -O2 does not reorder floating point.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ref_lbm.cpp")
OUT = os.path.join(HERE, "libref_lbm.so")


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "ref_lbm.h")]
    if not force and os.path.exists(OUT) and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in deps):
        return OUT
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", OUT, SRC]
    subprocess.check_call(cmd)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
