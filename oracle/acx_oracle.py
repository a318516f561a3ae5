"""ctypes view of oracle/acx_oracle.c — the plain single-threaded CPU decoder of FORMAT.md (§2).

ORACLE: test infrastructure, not product code.  It imports nothing from paper_2606_18900_b200."""
import ctypes
import os
import subprocess

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_lib = None

ERRORS = {0: "OK", -1: "E_MAGIC", -2: "E_VERSION", -3: "E_TRUNCATED", -4: "E_CORRUPT", -5: "E_RANGE", -6: "E_LEVEL",
          -7: "E_NOMEM"}

HEADER_FIELDS = ["N", "n_blocks", "n_segs", "log2_bs", "min_match", "W", "prob_bits", "n_tables", "max_level", "max_cmds",
                 "flags", "log2_seg", "q_min", "q_mode", "n_qpairs", "tables_off", "qtab_off", "blocktab_off", "dir_off",
                 "fnv_off", "payload_off", "archive_bytes", "total_lit", "total_match_bytes", "total_matches", "total_cmds",
                 "total_litq", "src_window"]


class OracleError(Exception):
    def __init__(self, rc):
        super().__init__(ERRORS.get(rc, str(rc)))
        self.code = rc
        self.name = ERRORS.get(rc, str(rc))


def build(force=False):
    src = os.path.join(_DIR, "acx_oracle.c")
    out = os.path.join(_DIR, "libacx_oracle.so")
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        subprocess.run(["gcc", "-O2", "-std=c11", "-Wall", "-shared", "-fPIC", "-o", out, src], check=True)
    return out


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        p, u64, u32 = ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint32
        _lib.acx_oracle_header.argtypes = [p, u64, p]
        _lib.acx_oracle_decode.argtypes = [p, u64, p, u64, ctypes.c_int]
        _lib.acx_oracle_decode_prefix.argtypes = [p, u64, p, u64, ctypes.c_int, u64]
        _lib.acx_oracle_block_segs.argtypes = [p, u64, u64, p]
        _lib.acx_oracle_segment.argtypes = [p, u64, u64] + [p] * 9
        _lib.acx_oracle_rans.argtypes = [p, u32, u32, p, p, u64, p, p, p, p, p]
        _lib.acx_oracle_fnv1a64.argtypes = [p, u64]
        _lib.acx_oracle_fnv1a64.restype = u64
    return _lib


def _arr(a):
    a = np.frombuffer(a, dtype=np.uint8) if isinstance(a, (bytes, bytearray)) else a
    return np.ascontiguousarray(a, dtype=np.uint8)


def header(archive):
    a = _arr(archive)
    f = np.zeros(len(HEADER_FIELDS), dtype=np.uint64)
    rc = _load().acx_oracle_header(a.ctypes.data, a.size, f.ctypes.data)
    if rc:
        raise OracleError(rc)
    return {k: int(v) for k, v in zip(HEADER_FIELDS, f)}


def decode(archive, check_levels=True):
    """The whole decompressed output (uint8 array).  Raises OracleError on any format violation."""
    a = _arr(archive)
    n = header(a)["N"]
    out = np.zeros(max(n, 1), dtype=np.uint8)
    rc = _load().acx_oracle_decode(a.ctypes.data, a.size, out.ctypes.data, n, 1 if check_levels else 0)
    if rc:
        raise OracleError(rc)
    return out[:n]


def decode_prefix(archive, n_blocks, check_levels=False, out=None):
    """The first n_blocks blocks (a prefix is self-sufficient: sources precede destinations)."""
    a = _arr(archive)
    h = header(a)
    n = min(h["N"], n_blocks << h["log2_bs"])
    out = np.zeros(max(n, 1), dtype=np.uint8) if out is None else out
    rc = _load().acx_oracle_decode_prefix(a.ctypes.data, a.size, out.ctypes.data, n, 1 if check_levels else 0, n_blocks)
    if rc:
        raise OracleError(rc)
    return out[:n]


def block_segs(archive, b):
    """(first segment, one past the last segment, level) of block b (FORMAT.md §1.4)."""
    a = _arr(archive)
    o = np.zeros(3, dtype=np.uint64)
    rc = _load().acx_oracle_block_segs(a.ctypes.data, a.size, b, o.ctypes.data)
    if rc:
        raise OracleError(rc)
    return int(o[0]), int(o[1]), int(o[2])


def segment(archive, sg):
    """Stage-level view of segment sg: dict of tokens, literals (in output order), sources, lengths and positions."""
    a = _arr(archive)
    lib = _load()
    counts = np.zeros(11, dtype=np.uint64)
    rc = lib.acx_oracle_segment(a.ctypes.data, a.size, sg, counts.ctypes.data, *([None] * 8))
    if rc:
        raise OracleError(rc)
    c = [int(v) for v in counts]
    n_cmd, n_match, n_lit = c[0], c[1], c[2] + c[3]
    r = dict(n_cmd=n_cmd, n_match=n_match, n_lit_a=c[2], n_lit_q=c[3], n_sym_q=c[4], n_lit=n_lit, n_words=c[5], n_ext=c[6],
             level=c[7], block=c[8], out_start=c[9], out_end=c[10],
             cmd=np.zeros(n_cmd, np.uint8), mlen=np.zeros(n_match, np.uint8), lit=np.zeros(n_lit, np.uint8),
             src=np.zeros(n_match, np.uint64), lit_len=np.zeros(n_cmd, np.uint32), match_len=np.zeros(n_cmd, np.uint32),
             lit_pos=np.zeros(n_cmd, np.uint32), out_pos=np.zeros(n_cmd, np.uint64))
    rc = lib.acx_oracle_segment(a.ctypes.data, a.size, sg, counts.ctypes.data, *[r[k].ctypes.data for k in
                                ("cmd", "mlen", "lit", "src", "lit_len", "match_len", "lit_pos", "out_pos")])
    if rc:
        raise OracleError(rc)
    return r


def rans_decode(freq, tid, states, streams, prob_bits=11):
    """FORMAT.md §1.7 alone.  freq: (n_tables, n_sym) u16; tid: table id per symbol; states: 32 u32; streams: 32 lists of
    u16 words (state k's own stream); prob_bits: one value or one per table.  Returns (symbol indices, final_states,
    words_used[32])."""
    freq = np.ascontiguousarray(freq, dtype=np.uint16)
    freq = freq.reshape(1, -1) if freq.ndim == 1 else freq
    pb = np.ascontiguousarray(np.broadcast_to(np.asarray(prob_bits, dtype=np.uint32), (freq.shape[0],)))
    tid = np.ascontiguousarray(tid, dtype=np.uint8)
    st = np.ascontiguousarray(states, dtype=np.uint32).copy()
    assert len(streams) == 32
    off = np.zeros(33, dtype=np.uint64)
    off[1:] = np.cumsum([len(s) for s in streams])
    w = np.ascontiguousarray(np.concatenate([np.asarray(s, dtype="<u2") for s in streams] + [np.zeros(1, "<u2")]))
    sym = np.zeros(max(tid.size, 1), dtype=np.uint16)
    used = np.zeros(32, dtype=np.uint64)
    rc = _load().acx_oracle_rans(freq.ctypes.data, freq.shape[0], freq.shape[1], pb.ctypes.data, tid.ctypes.data, tid.size,
                                 st.ctypes.data, w.ctypes.data, off.ctypes.data, sym.ctypes.data, used.ctypes.data)
    if rc:
        raise OracleError(rc)
    return sym[:tid.size], st, used.astype(np.int64)


def fnv1a64(data):
    a = _arr(data)
    return int(_load().acx_oracle_fnv1a64(a.ctypes.data, a.size))
