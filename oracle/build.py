"""Build the CPU oracle shared library (TEST INFRASTRUCTURE, see mpcd_oracle.c).

    python oracle/build.py

Compiles oracle/mpcd_oracle.c with gcc into oracle/libmpcd_oracle.so.  Flags:
-O2 -ffp-contract=off (no FMA contraction: streaming and binning are defined as
separately rounded operations, SURVEY.md 8c readings A6/A7), never -ffast-math.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mpcd_oracle.c")
INC = os.path.join(HERE, "mpcd_oracle_steps.inc")
LIB = os.path.join(HERE, "libmpcd_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB):
        if os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(INC)):
            return LIB
    cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
