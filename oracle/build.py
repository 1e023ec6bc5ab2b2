"""Build the CPU oracle shared library (test infrastructure; see xpr_oracle.h).

    python oracle/build.py          # -> oracle/libxpr_oracle.so

Flags follow DESIGN.md rule R1: no FMA contraction, no fast-math, so that every fp32 operation
of the parity mode is individually rounded in the documented order.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "xpr_oracle.cpp")
OUT = os.path.join(HERE, "libxpr_oracle.so")
FLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
         "-Wall", "-Wextra", "-Wno-unused-parameter"]


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "xpr_oracle_ray.inc"), os.path.join(HERE, "xpr_oracle_feat.inc"), os.path.join(HERE, "xpr_oracle_lin.inc"), os.path.join(HERE, "xpr_oracle.h"), os.path.abspath(__file__)]
    if not force and os.path.exists(OUT) and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in deps):
        return OUT
    cmd = ["g++", *FLAGS, "-o", OUT, SRC]
    subprocess.run(cmd, check=True)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
