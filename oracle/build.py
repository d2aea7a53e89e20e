"""Build the CPU oracle (test infrastructure) into oracle/libref_lbm.so.

    python oracle/build.py

-ffp-contract=off: the compiler contracts nothing, so ref_lbm.cpp has exactly the fused
multiply-adds it spells out as std::fma and every other operation is one IEEE-754
rounding.  -O2 does not reorder floating point.  -mfma (when the
host CPU has it) only turns the std::fma calls into one instruction instead of a libm
call; the result is the same correctly rounded value either way.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ref_lbm.cpp")
OUT = os.path.join(HERE, "libref_lbm.so")


def _host_has_fma() -> bool:
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("flags"):
                    return " fma " in line + " "
    except OSError:
        pass
    return False


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "ref_lbm.h")]
    if not force and os.path.exists(OUT) and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in deps):
        return OUT
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-Wall", "-Wextra"] + (["-mfma"] if _host_has_fma() else []) + ["-o", OUT, SRC]
    subprocess.check_call(cmd)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
