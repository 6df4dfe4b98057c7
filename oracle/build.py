"""Build oracle/liboracle.so from oracle/mhd_oracle.c (TEST INFRASTRUCTURE).

Plain gcc, fp64, no fast-math, no FMA contraction.
Run as `python oracle/build.py` or call `build()`.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mhd_oracle.c")
LIB = os.path.join(HERE, "liboracle.so")

FLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-std=c99",
         "-shared", "-fPIC", "-Wall", "-Wno-misleading-indentation"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc"] + FLAGS + ["-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
