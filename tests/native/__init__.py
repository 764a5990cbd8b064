"""Test-side native helpers (never imported by the product)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "curand_philox_check.cu")
_LIB = os.path.join(_HERE, "libcurand_philox_check.so")


def build(force: bool = False) -> str:
    """nvcc cross-compiles for sm_100a without a GPU; __graft_entry__.build() calls this too."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_SRC) > os.path.getmtime(_LIB):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call([nvcc, "-O2", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC",
                               "-shared", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def curand_philox(key, ctr) -> np.ndarray:
    """The toolkit's curand_Philox4x32_10 on the GPU: key (2,), ctr (n, 4) uint32 -> (n, 4) uint32."""
    L = C.CDLL(build())
    L.curand_philox4x32_10_host.restype = C.c_int
    L.curand_philox4x32_10_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
    k = np.ascontiguousarray(key, dtype=np.uint32)
    c = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    out = np.zeros_like(c)
    rc = L.curand_philox4x32_10_host(k.ctypes.data, c.ctypes.data, out.ctypes.data, len(c))
    if rc:
        raise RuntimeError("curand_philox4x32_10_host: cudaError %d" % rc)
    return out
