"""ctypes binding of encoder.cpp: writes ACX-B200 archives (FORMAT.md).  Produces test inputs only."""
import ctypes

import numpy as np

_lib = None


class EncOpts(ctypes.Structure):
    _fields_ = [("log2_bs", ctypes.c_uint32), ("min_match", ctypes.c_uint32), ("max_level", ctypes.c_uint32),
                ("threads", ctypes.c_uint32), ("src_window", ctypes.c_uint64), ("chunk_log2", ctypes.c_uint32),
                ("batch_chunks", ctypes.c_uint32), ("chain_depth", ctypes.c_uint32), ("hash_log2", ctypes.c_uint32),
                ("with_fnv", ctypes.c_uint32), ("log2_seg", ctypes.c_uint32), ("q_min", ctypes.c_uint32), ("q_mode", ctypes.c_uint32)]


def _load():
    global _lib
    if _lib is None:
        from ..build import build_encoder
        _lib = ctypes.CDLL(build_encoder())
        _lib.acx_enc_default_opts.argtypes = [ctypes.POINTER(EncOpts)]
        _lib.acx_encode.argtypes = [ctypes.c_void_p, ctypes.c_uint64, ctypes.POINTER(EncOpts),
                                    ctypes.POINTER(ctypes.c_void_p), ctypes.POINTER(ctypes.c_uint64)]
        _lib.acx_encode.restype = ctypes.c_int
        _lib.acx_enc_free.argtypes = [ctypes.c_void_p]
    return _lib


def encode(data, block_size=16384, **kw):
    """data: uint8 numpy array (or bytes).  Returns the archive as a uint8 numpy array.

    Options (encoder.cpp acx_enc_opts): min_match, max_level (default 2), threads, src_window, chunk_log2, batch_chunks,
    chain_depth, hash_log2, with_fnv, log2_seg (segment size, default min(block, 16 KB)), q_min (literal runs of this many
    bytes or more form the stream LITQ; default 64, 0 = one literal class), q_mode (0 bytes, 1 pairs = default, 2 = the smaller)."""
    lib = _load()
    data = np.ascontiguousarray(np.frombuffer(data, dtype=np.uint8) if isinstance(data, (bytes, bytearray)) else data)
    assert data.dtype == np.uint8
    o = EncOpts()
    lib.acx_enc_default_opts(ctypes.byref(o))
    lb = int(block_size).bit_length() - 1
    assert 1 << lb == block_size, "block_size must be a power of two"
    o.log2_bs = lb
    for k, v in kw.items():
        setattr(o, k, v)
    out, n = ctypes.c_void_p(), ctypes.c_uint64()
    rc = lib.acx_encode(data.ctypes.data, data.size, ctypes.byref(o), ctypes.byref(out), ctypes.byref(n))
    if rc:
        raise RuntimeError("acx_encode failed: %d" % rc)
    try:
        return np.ctypeslib.as_array(ctypes.cast(out, ctypes.POINTER(ctypes.c_uint8)), (n.value,)).copy()
    finally:
        lib.acx_enc_free(out)
