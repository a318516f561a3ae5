"""ctypes view of oracle/acx_mt.c — the multithreaded CPU decoder used as a reported baseline (BASELINE.json north_star).

CPU BASELINE: measurement infrastructure, not product code.  It imports nothing from paper_2606_18900_b200."""
import ctypes
import os
import subprocess

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_lib = None


def build(force=False):
    src = os.path.join(_DIR, "acx_mt.c")
    out = os.path.join(_DIR, "libacx_mt.so")
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        subprocess.run(["gcc", "-O2", "-std=c11", "-Wall", "-shared", "-fPIC", "-pthread", "-o", out, src], check=True)
    return out


def decode(archive, threads=None, out=None):
    """The whole decompressed output, decoded by `threads` host threads (default: all cores)."""
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.acx_mt_decode.argtypes = [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int]
    a = np.ascontiguousarray(np.frombuffer(archive, dtype=np.uint8) if isinstance(archive, (bytes, bytearray)) else archive)
    n = int(a[16:24].view(np.uint64)[0])
    out = np.zeros(max(n, 1), dtype=np.uint8) if out is None else out
    rc = _lib.acx_mt_decode(a.ctypes.data, a.size, out.ctypes.data, out.size, threads or os.cpu_count() or 1)
    if rc:
        raise RuntimeError("acx_mt_decode failed: %d" % rc)
    return out[:n]
