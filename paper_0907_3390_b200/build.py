"""Build the CUDA library (the product) in-tree: paper_0907_3390_b200/libgamer_hydro.so, sm_100a only.

`python -m paper_0907_3390_b200.build [--ptxas-v]` always rebuilds (build() itself skips an up-to-date library).  nvcc cross-compiles without a GPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = [os.path.join(CSRC, "gamer_hydro.cu")]
DEPS = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC))] + \
    [os.path.join(os.path.dirname(HERE), "include", f) for f in ("gamer_hydro.h", "gamer_probes.h")]
LIB = os.path.join(HERE, "libgamer_hydro.so")
# the measurement aids of bench.py (include/gamer_probes.h) are a library of their own, not part of the product ABI
PROBE_SOURCES = [os.path.join(CSRC, "probes.cu")]
PROBE_LIB = os.path.join(HERE, "libgamer_probes.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "-cudart", "shared"]


def nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _compile(lib, sources, force, verbose, extra):
    if (not force) and os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in DEPS):
        return lib
    tmp = lib + ".tmp%d" % os.getpid()          # per process: concurrent builders do not collide
    cmd = [nvcc()] + NVCC_FLAGS + list(extra) + ["-o", tmp] + sources
    if verbose:
        print(" ".join(cmd), file=sys.stderr)
    subprocess.run(cmd, check=True)
    os.replace(tmp, lib)
    return lib


def build(force=False, verbose=False, extra=(), out=None):
    """Compile the product library to `out` (default: the in-tree libgamer_hydro.so) and, for the default target, the
    probe library beside it; `extra` = more nvcc flags.  Returns the path of the product library."""
    lib = _compile(out or LIB, SOURCES, force, verbose, extra)
    if out is None:
        _compile(PROBE_LIB, PROBE_SOURCES, force, verbose, ())
    return lib


if __name__ == "__main__":
    print(build(force=True, verbose=True,
                extra=["-Xptxas", "-v"] if "--ptxas-v" in sys.argv else []))
