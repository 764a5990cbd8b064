"""Build step: compile the CUDA library in-tree for sm_100a (nvcc cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libptglass.so")
SOURCES = [os.path.join(CSRC, "ptglass.cu"), os.path.join(CSRC, "microbench.cu")]
DEPS = SOURCES + sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cuh")) + [
    os.path.join(os.path.dirname(_HERE), "include", "ptglass.h"), os.path.join(os.path.dirname(_HERE), "include", "ptglass_diag.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


STAMP = LIB + ".flags"


def _dev_flags():
    """PTG_DEV_LATTICE="d,log2L" (development only): compile the kernels for that one fast lattice (+ the general path
    of the same d), which takes a quarter of the time of the full build.  The flags of the last build are kept in a stamp
    file, so a later build without the variable rebuilds the full library."""
    v = os.environ.get("PTG_DEV_LATTICE", "")
    if not v:
        return []
    d, lg = (int(x) for x in v.split(","))
    return ["-DPTG_DEV_D=%d" % d, "-DPTG_DEV_LG=%d" % lg] + os.environ.get("PTG_DEV_EXTRA", "").split()


def build(force: bool = False, verbose: bool = False) -> str:
    flags = NVCC_FLAGS + _dev_flags()
    old = open(STAMP).read() if os.path.exists(STAMP) else ""
    stale = (not os.path.exists(LIB)) or old != " ".join(flags) or any(
        os.path.getmtime(p) > os.path.getmtime(LIB) for p in DEPS)
    if force or stale:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB + ".tmp%d" % os.getpid()
        cmd = [nvcc] + flags + ["-o", tmp] + SOURCES
        out = subprocess.run(cmd, capture_output=True, text=True)
        if out.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + out.stdout + out.stderr)
        os.replace(tmp, LIB)
        with open(STAMP, "w") as f:
            f.write(" ".join(flags))
        with open(os.path.join(_HERE, "build.log"), "w") as f:
            f.write(" ".join(cmd) + "\n" + out.stdout + out.stderr)
        if verbose:
            print(out.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
