"""Build libastra_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libastra_b200.so")
LIB_DIAG = os.path.join(_HERE, "libastra_b200_diag.so")      # same sources with -DASTRA_DIAG (per-stage clocks)
SOURCES = ["astra_engine.cu", "astra_loader.cpp", "astra_api.cpp"]
HEADERS = ["astra_internal.h", os.path.join("..", "..", "include", "astra.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall", "-diag-suppress", "550"]


def _nvcc() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.sep not in p or os.path.exists(p)):
            return p
    return "nvcc"


def needs_build(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, diag: bool = False) -> str:
    """The product library (default), or the instrumented one (diag=True: -DASTRA_DIAG adds per-stage SM
    clock counters read by astra_read_diag; never used for a timing that is reported as a result)."""
    lib = LIB_DIAG if diag else LIB
    # experiments: ASTRA_EXTRA_DEFS="-DX -DY" ASTRA_LIB_SUFFIX=_x builds libastra_b200_x.so with those defines
    extra = os.environ.get("ASTRA_EXTRA_DEFS", "").split()
    suffix = os.environ.get("ASTRA_LIB_SUFFIX", "")
    if suffix:
        lib = os.path.join(_HERE, f"libastra_b200{suffix}.so")
    if not force and not needs_build(lib):
        return lib
    objs = []
    for s in SOURCES:
        o = os.path.join(CSRC, os.path.splitext(s)[0] + suffix + (".diag.o" if diag else ".o"))
        cmd = [_nvcc()] + NVCC_FLAGS + extra + (["-DASTRA_DIAG"] if diag else []) + (["-Xptxas", "-v"] if verbose else []) + \
              ["-x", "cu", "-c", os.path.join(CSRC, s), "-o", o]
        subprocess.check_call(cmd)
        objs.append(o)
    tmp = lib + f".tmp{os.getpid()}"
    subprocess.check_call([_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + objs)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose=True, diag="--diag" in sys.argv))
