"""Build the CPU oracle shared library (test infrastructure only).

    python oracle/build.py

-ffp-contract=off: every fp64 operation rounds once, as written (reading R17).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sfh_oracle.cpp")
LIB = os.path.join(HERE, "libsfh_oracle.so")
LIB16 = os.path.join(HERE, "libsfh_oracle16.so")    # the same source with blocks of 16^3 cells


def lib_path(ncell=8):
    return LIB16 if ncell == 16 else LIB


def build(force=False, ncell=8):
    out = lib_path(ncell)
    if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(SRC):
        return out
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-DSFH_ORACLE_N=%d" % ncell, "-o", out, SRC]
    subprocess.run(cmd, check=True)
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv), build(force="--force" in sys.argv, ncell=16))
