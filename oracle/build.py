"""Build oracle/libsco.so (the fp64 CPU oracle; TEST INFRASTRUCTURE, see oracle/sco.h).

Run as `python oracle/build.py` or call `build()`; rebuilds only when sco.cpp / sco.h are newer.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libsco.so")
SRC = [os.path.join(HERE, "sco.cpp"), os.path.join(HERE, "sco.h")]
# -ffp-contract=off: the inclusion test is specified without FMA contraction (R4).
CMD = ["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
       "-Wall", "-Wextra", SRC[0], "-o", LIB]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(s) for s in SRC)):
        return LIB
    subprocess.run(CMD, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
