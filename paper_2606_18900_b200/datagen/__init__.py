"""ctypes binding of datagen.c: seeded synthetic FASTQ / FASTA inputs.

Shared by the oracle-side and the CUDA-side tests; contains none of the method's arithmetic."""
import ctypes
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_lib = None


def _load():
    global _lib
    if _lib is None:
        from ..build import build_datagen
        _lib = ctypes.CDLL(build_datagen())
        u64, p = ctypes.c_uint64, ctypes.c_void_p
        _lib.acx_gen_fastq.argtypes = [u64, u64, u64, u64, u64, p]
        _lib.acx_gen_fastq.restype = ctypes.c_int
        _lib.acx_fastq_n_reads.argtypes = [u64]
        _lib.acx_fastq_n_reads.restype = u64
        _lib.acx_fastq_index.argtypes = [u64, u64, u64, p]
        _lib.acx_fastq_index.restype = ctypes.c_int
        _lib.acx_gen_fasta.argtypes = [u64, u64, p]
        _lib.acx_gen_fasta.restype = ctypes.c_int
        _lib.acx_gen_region_index.argtypes = [u64, u64, u64, u64, p]
        _lib.acx_gen_region_index.restype = ctypes.c_int
    return _lib


def fastq(seed, n_bytes, ref_len, lo=0, hi=None, threads=None):
    """Bytes [lo, hi) of the synthetic FASTQ file of n_bytes bytes (configs[0], [1], [4])."""
    lib = _load()
    hi = n_bytes if hi is None else hi
    out = np.empty(hi - lo, dtype=np.uint8)
    threads = threads or min(os.cpu_count() or 1, 32)
    step = max(1 << 20, -(-(hi - lo) // threads))
    parts = [(a, min(a + step, hi)) for a in range(lo, hi, step)]

    def run(ab):
        a, b = ab
        rc = lib.acx_gen_fastq(seed, ref_len, n_bytes, a, b, out[a - lo:].ctypes.data)
        if rc:
            raise ValueError("acx_gen_fastq failed")
    if len(parts) <= 1:
        for ab in parts:
            run(ab)
    else:
        with ThreadPoolExecutor(threads) as ex:
            list(ex.map(run, parts))
    return out


def fastq_n_reads(n_bytes):
    return int(_load().acx_fastq_n_reads(n_bytes))


def fastq_index(n_bytes, first=0, count=None):
    """FORMAT.md §4 index entries (offset | len << 40) of the whole reads of the FASTQ file."""
    lib = _load()
    count = fastq_n_reads(n_bytes) - first if count is None else count
    out = np.empty(count, dtype=np.uint64)
    if lib.acx_fastq_index(n_bytes, first, count, out.ctypes.data):
        raise ValueError("acx_fastq_index failed")
    return out


def fasta(seed, n_bytes):
    """The synthetic genome FASTA of exactly n_bytes bytes (configs[2], [3])."""
    out = np.empty(n_bytes, dtype=np.uint8)
    if _load().acx_gen_fasta(seed, n_bytes, out.ctypes.data):
        raise ValueError("acx_gen_fasta failed")
    return out


def region_index(seed, n_bytes, n, length=150):
    """n index entries of fixed-length regions at uniform offsets (configs[2]: 10^6 x 150 B)."""
    out = np.empty(n, dtype=np.uint64)
    if _load().acx_gen_region_index(seed, n_bytes, n, length, out.ctypes.data):
        raise ValueError("acx_gen_region_index failed")
    return out
