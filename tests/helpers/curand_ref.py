"""Builds and calls tests/helpers/curand_philox_host.cu (cuRAND's Philox4x32-10, host path)."""
import ctypes as C
import os
import shutil
import subprocess
import tempfile

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "curand_philox_host.cu")
_lib = None


def available():
    return shutil.which("nvcc") is not None or os.path.exists("/usr/local/cuda/bin/nvcc")


def _load():
    global _lib
    if _lib is None:
        nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
        out = os.path.join(tempfile.gettempdir(), "cg_curand_philox_host_%d.so" % os.getuid())
        subprocess.check_call([nvcc, "-O2", "-shared", "-Xcompiler", "-fPIC", "-cudart", "static",
                               "-o", out, _SRC])
        _lib = C.CDLL(out)
        _lib.curand_philox_batch.restype = None
        _lib.curand_philox_batch.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
    return _lib


def philox_batch(ctr, key):
    ctr = np.ascontiguousarray(ctr, np.uint32).reshape(-1, 4)
    key = np.ascontiguousarray(key, np.uint32).reshape(-1, 2)
    out = np.empty_like(ctr)
    _load().curand_philox_batch(ctr.shape[0], ctr.ctypes.data, key.ctypes.data, out.ctypes.data)
    return out
