"""Builds libiris_so.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2607_01338_b200.build [--force] [--verbose]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libiris_so.so")
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def sources():
    return [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cu", ".cuh", ".inc"))] + [
        os.path.join(os.path.dirname(HERE), "include", "iris_so.h")]


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in sources())


LIB_CHECKED = os.path.join(HERE, "libiris_so_checked.so")


def build(force=False, verbose=False, checked=False):
    """Compile csrc/iris_so.cu -> libiris_so.so (checked: -> libiris_so_checked.so with -DIRIS_SO_CHECKED, the
    bounds-checked build tests/test_sanitizers.py runs). Returns the library path."""
    lib = LIB_CHECKED if checked else LIB
    if not force and os.path.exists(lib) and all(os.path.getmtime(s) <= os.path.getmtime(lib) for s in sources()):
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = lib + ".tmp%d" % os.getpid()
    cmd = ([nvcc] + NVCC_FLAGS + (["-DIRIS_SO_CHECKED"] if checked else []) + (["-Xptxas", "-v"] if verbose else [])
           + ["-o", tmp, os.path.join(CSRC, "iris_so.cu")])
    subprocess.run(cmd, check=True)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, checked="--checked" in sys.argv))
