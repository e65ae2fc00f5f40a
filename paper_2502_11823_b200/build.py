"""Builds ``libsft_b200.so`` (the C-ABI library of include/sft.h) in-tree with nvcc for sm_100a.

    python -m paper_2502_11823_b200.build [--force]

The shared library is written next to this file so that it travels with the source tree (it is
git-ignored).  nvcc cross-compiles without a GPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsft_b200.so")
SOURCES = [os.path.join(CSRC, "sft_lib.cu")]


def deps():
    """Everything the library is compiled from: every file under csrc/ (sources, headers, generated coefficient tables)
    and the public header."""
    import glob
    return sorted(glob.glob(os.path.join(CSRC, "*"))) + [os.path.join(os.path.dirname(HERE), "include", "sft.h")]


NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
              "-cudart", "static"]


def nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    raise RuntimeError("nvcc not found")


def up_to_date():
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(d) <= t for d in deps())


def build(force=False, verbose=False, extra=()):
    """Compiles the library if it is missing or older than its sources.  Returns its path."""
    if not force and up_to_date():
        return LIB
    extra = list(extra) + os.environ.get("SFT_NVCC_EXTRA", "").split()      # e.g. -DSFT_MINB=4
    cmd = [nvcc()] + NVCC_FLAGS + extra + ["-o", LIB] + SOURCES
    if verbose:
        print(" ".join(cmd), flush=True)
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    if verbose and (r.stdout or r.stderr):
        print(r.stdout + r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True,
                extra=["-Xptxas", "-v"] if "--ptxas-v" in sys.argv else ()))
