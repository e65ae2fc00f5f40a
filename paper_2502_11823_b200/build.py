"""Builds ``libsft_b200.so`` (the C-ABI library of include/sft.h) in-tree with nvcc for sm_100a.

    python -m paper_2502_11823_b200.build [--force] [--checked]

``--checked`` builds the same library with -DSFT_CHECKED: every indexed global access of the main path is tested against the
extent of its buffer and a call whose kernel tripped a test returns SFT_ECUDA (sft_kernels.cuh, SFT_CHK).  For running the GPU
tests once after a change of the index arithmetic; slower, never the library that is timed.  ``sft_version()`` says which one
is loaded.

The shared library is written next to this file so that it travels with the source tree (it is
git-ignored).  nvcc cross-compiles without a GPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsft_b200.so")
SOURCES = [os.path.join(CSRC, f) for f in ("sft_lib.cu", "sft_var_bns.cu", "sft_var_misc.cu", "sft_var_lisa.cu", "sft_var_any1.cu", "sft_var_any2.cu", "sft_var_any3.cu",
                                             "sft_var_any4.cu")]
OBJ = os.path.join(HERE, "_obj")


def deps():
    """Everything the library is compiled from: every file under csrc/ (sources, headers, generated coefficient tables)
    and the public header."""
    import glob
    return sorted(glob.glob(os.path.join(CSRC, "*"))) + [os.path.join(os.path.dirname(HERE), "include", "sft.h")]


NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]


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
    """Compiles the library if it is missing or older than its sources.  The variants of the fused kernel are spread over
    several translation units, compiled side by side (one nvcc process each), then linked.  Returns the library's path."""
    if not force and up_to_date():
        return LIB
    extra = list(extra) + os.environ.get("SFT_NVCC_EXTRA", "").split()      # e.g. -DSFT_MINB=4
    os.makedirs(OBJ, exist_ok=True)
    procs = []
    for src in SOURCES:
        obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")
        cmd = [nvcc()] + NVCC_FLAGS + extra + ["-c", "-o", obj, src]
        if verbose:
            print(" ".join(cmd), flush=True)
        procs.append((obj, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    objs, log, bad = [], "", False
    for obj, pr in procs:
        out, _ = pr.communicate()
        log += out
        bad |= pr.returncode != 0
        objs.append(obj)
    if bad:
        raise RuntimeError("nvcc failed:\n" + log)
    cmd = [nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static", "-o", LIB] + objs
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + r.stdout + r.stderr)
    if verbose and log:
        print(log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv or "--checked" in sys.argv, verbose=True,
                extra=(["-Xptxas", "-v"] if "--ptxas-v" in sys.argv else []) + (["-DSFT_CHECKED"] if "--checked" in sys.argv else [])))
