"""Build libsc.so (the C-ABI library of include/sc.h) for sm_100a with nvcc, in-tree.

    python -m paper_1409_4441_b200.build        # or build() from Python

nvcc cross-compiles without a GPU.  The .so sits next to this file so that it travels with the
repository snapshot to the GPU box (it is git-ignored).
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libsc.so")
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["sc_plan.cu", "sc_generic.cu", "sc_fast.cu", "sc_belt.cu", "sc_nested.cu"]
HEADERS = [os.path.join(CSRC, "sc_internal.cuh"), os.path.join(CSRC, "sc_fast.cuh"), os.path.join(ROOT, "include", "sc.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         # fp64 inclusion test is specified without FMA contraction on the host side as well
         "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall", "-shared", "-cudart", "static"]


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
