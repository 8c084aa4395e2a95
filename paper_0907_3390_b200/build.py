"""Build the CUDA library (the product) in-tree: paper_0907_3390_b200/libgamer_hydro.so, sm_100a only.

`python -m paper_0907_3390_b200.build [--force] [--verbose]`.  nvcc cross-compiles without a GPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = [os.path.join(CSRC, "gamer_hydro.cu")]
DEPS = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC))] + \
    [os.path.join(os.path.dirname(HERE), "include", "gamer_hydro.h")]
LIB = os.path.join(HERE, "libgamer_hydro.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "-cudart", "shared"]


def nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def build(force=False, verbose=False, extra=(), out=None):
    """Compile the library to `out` (default: the in-tree libgamer_hydro.so); `extra` = more nvcc flags."""
    lib = out or LIB
    if (not force) and os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in DEPS):
        return lib
    tmp = lib + ".tmp%d" % os.getpid()          # per process: concurrent builders do not collide
    cmd = [nvcc()] + NVCC_FLAGS + list(extra) + ["-o", tmp] + SOURCES
    if verbose:
        print(" ".join(cmd), file=sys.stderr)
    subprocess.run(cmd, check=True)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv or True, verbose=True,
                extra=["-Xptxas", "-v"] if "--ptxas-v" in sys.argv else []))
