"""Build libsc.so (the C-ABI library of include/sc.h) for sm_100a with nvcc, in-tree.

    python -m paper_1409_4441_b200.build        # or build() from Python

nvcc cross-compiles without a GPU.  The .so sits next to this file so that it travels with the
repository snapshot to the GPU box (it is git-ignored).  Every source file is compiled to an object
of its own (in parallel, only when stale) and the objects are linked into the library.
"""
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libsc.so")
CSRC = os.path.join(HERE, "csrc")
OBJDIR = os.path.join(HERE, "build")
SOURCES = ["sc_plan.cu", "sc_generic.cu", "sc_fast.cu", "sc_sym_b1.cu", "sc_sym_bn.cu", "sc_sym_pl.cu", "sc_sym_pair.cu", "sc_belt.cu", "sc_nested.cu", "sc_probe.cu", "sc_static.cu"]
HEADERS = [os.path.join(CSRC, "sc_internal.cuh"), os.path.join(CSRC, "sc_fast.cuh"), os.path.join(CSRC, "sc_sym.cuh"), os.path.join(ROOT, "include", "sc.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
CFLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
          # fp64 inclusion test is specified without FMA contraction on the host side as well
          "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall"]
LFLAGS = ["-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a"]


def _mtime(p):
    return os.path.getmtime(p) if os.path.exists(p) else -1.0


def _obj(src):
    return os.path.join(OBJDIR, os.path.splitext(src)[0] + ".o")


def build(force: bool = False, verbose: bool = False) -> str:
    common = max(_mtime(h) for h in HEADERS + [os.path.abspath(__file__)])
    stale = [s for s in SOURCES
             if force or _mtime(_obj(s)) < max(common, _mtime(os.path.join(CSRC, s)))]
    if not stale and _mtime(LIB) >= max(_mtime(_obj(s)) for s in SOURCES):
        return LIB
    os.makedirs(OBJDIR, exist_ok=True)

    def compile_one(src):
        cmd = [NVCC] + CFLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-c", os.path.join(CSRC, src), "-o", _obj(src)]
        subprocess.run(cmd, check=True, cwd=HERE)

    with ThreadPoolExecutor(max_workers=max(1, min(len(stale), os.cpu_count() or 1))) as ex:
        list(ex.map(compile_one, stale))
    subprocess.run([NVCC] + LFLAGS + [_obj(s) for s in SOURCES] + ["-o", LIB], check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
