"""ctypes view of oracle/acx_rans_rows.c — the plain C rANS row encoder / decoder of the entropy micro-benchmark.

ORACLE: test infrastructure, not product code.  It imports nothing from paper_2606_18900_b200."""
import ctypes
import os
import subprocess

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_lib = None


def build(force=False):
    src = os.path.join(_DIR, "acx_rans_rows.c")
    out = os.path.join(_DIR, "libacx_rans_rows.so")
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        subprocess.run(["gcc", "-O2", "-std=c11", "-Wall", "-shared", "-fPIC", "-o", out, src], check=True)
    return out


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        p, u64 = ctypes.c_void_p, ctypes.c_uint64
        _lib.acx_rows_encode.argtypes = [p, u64, u64, p, p, u64, p]
        _lib.acx_rows_decode.argtypes = [p, u64, u64, u64, p, p, p]
    return _lib


def row_capacity(row_bytes):
    return (256 + 2 * row_bytes + 15) // 16 * 16


def encode(rows, freq):
    """rows: (n_rows, row_bytes) uint8; freq: 256 frequencies summing to 2^11.  Returns (encoded (n_rows, cap) uint8, sizes)."""
    rows = np.ascontiguousarray(rows, dtype=np.uint8)
    freq = np.ascontiguousarray(freq, dtype=np.uint16)
    n, rb = rows.shape
    cap = row_capacity(rb)
    out = np.zeros((n, cap), dtype=np.uint8)
    sizes = np.zeros(n, dtype=np.uint32)
    rc = _load().acx_rows_encode(rows.ctypes.data, n, rb, freq.ctypes.data, out.ctypes.data, cap, sizes.ctypes.data)
    if rc:
        raise ValueError("acx_rows_encode failed: %d" % rc)
    return out, sizes


def decode(enc, sizes, row_bytes, freq):
    enc = np.ascontiguousarray(enc, dtype=np.uint8)
    sizes = np.ascontiguousarray(sizes, dtype=np.uint32)
    freq = np.ascontiguousarray(freq, dtype=np.uint16)
    n, cap = enc.shape
    out = np.zeros((n, row_bytes), dtype=np.uint8)
    rc = _load().acx_rows_decode(enc.ctypes.data, n, row_bytes, cap, sizes.ctypes.data, freq.ctypes.data, out.ctypes.data)
    if rc:
        raise ValueError("acx_rows_decode failed: %d" % rc)
    return out
