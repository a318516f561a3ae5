"""Thin ctypes binding of include/aceapex.h (argument marshalling only: every step of the path runs in the CUDA
library).  torch is used for device memory and streams.  Fails loudly when the CUDA library is missing."""
import ctypes
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
_lib = None

ERRORS = {0: "OK", -1: "E_MAGIC", -2: "E_VERSION", -3: "E_TRUNCATED", -4: "E_CORRUPT", -5: "E_RANGE", -6: "E_BUDGET",
          -7: "E_WORKSPACE", -8: "E_CUDA", -9: "E_ARG", -10: "E_TOO_LARGE"}


class AceapexError(RuntimeError):
    def __init__(self, rc, what=""):
        self.code = rc
        self.name = ERRORS.get(rc, str(rc))
        super().__init__("%s%s" % (self.name, (": " + what) if what else ""))


class Info(ctypes.Structure):
    _fields_ = [(k, ctypes.c_uint64) for k in ("raw_bytes", "archive_bytes", "n_blocks", "block_size", "total_lit_bytes",
                                               "total_match_bytes", "total_matches", "total_cmds", "workspace_bytes",
                                               "n_segments", "total_litq_bytes")] + \
               [(k, ctypes.c_uint32) for k in ("max_level", "offset_width", "min_match", "max_cmds", "n_coded_planes",
                                               "has_fnv", "resident_warps", "segment_size", "q_min", "q_mode")]


class StreamStats(ctypes.Structure):
    _fields_ = [(k, ctypes.c_uint64) for k in ("n_windows", "n_slots", "bytes", "bad_blocks", "peak_device_bytes")] + \
               [(k, ctypes.c_float) for k in ("device_ms", "min_window_gbs", "max_window_gbs")] + [("reserved", ctypes.c_uint32)]


WINDOW_FN = ctypes.CFUNCTYPE(ctypes.c_int32, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_void_p, ctypes.c_void_p)


def lib_path():
    return os.path.join(_PKG, "libaceapex.so")


def load():
    """Loads libaceapex.so (built in-tree by paper_2606_18900_b200.build).  No fallback: raises if it is missing."""
    global _lib
    if _lib is None:
        path = lib_path()
        if not os.path.exists(path):
            raise ImportError("libaceapex.so is not built: run `python -m paper_2606_18900_b200.build cuda`")
        L = ctypes.CDLL(path)
        p, u64, u32, i32 = ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int32
        sig = {
            "aceapex_open": ([p, u64, p, ctypes.POINTER(p)], i32),
            "aceapex_close": ([p], i32),
            "aceapex_info": ([p, ctypes.POINTER(Info)], i32),
            "aceapex_set_workspace": ([p, p, u64], i32),
            "aceapex_set_stream": ([p, p], i32),
            "aceapex_decode_all": ([p, p], i32),
            "aceapex_decode_all_flags": ([p, p], i32),
            "aceapex_decode_all_fused": ([p, p], i32),
            "aceapex_decode_range": ([p, u64, u64, p, u64], i32),
            "aceapex_decode_reads": ([p, p, u64, p, u64, p], i32),
            "aceapex_decode_stream": ([p, u64, u64, p, u64, u64, WINDOW_FN, p, u64, ctypes.POINTER(StreamStats)], i32),
            "aceapex_reads_bytes": ([p, u64, p, u64, ctypes.POINTER(u64), p], i32),
            "aceapex_set_resident": ([p, u32, u64, u64, p], i32),
            "aceapex_verify_fnv": ([p, p, u64, u64, ctypes.POINTER(u64)], i32),
            "aceapex_decode_all_host": ([p, p, p, p], i32),
            "aceapex_check": ([p], i32),
            "aceapex_device_flags": ([p], u32),
            "aceapex_last_cuda_error": ([p], i32),
            "aceapex_strerror": ([i32], ctypes.c_char_p),
            "aceapex_launch_count": ([p], u64),
            "aceapex_graph_launch_count": ([p], u64),
            "aceapex_rans_row_capacity": ([u64], u64),
            "aceapex_rans_table_bytes": ([], u64),
            "aceapex_rans_scratch_bytes": ([u64], u64),
            "aceapex_rans_tables": ([p, p, p], i32),
            "aceapex_rans_encode": ([p, u64, u64, p, p, u64, p, p, u64, p], i32),
            "aceapex_rans_decode": ([p, u64, u64, u64, p, p, p, p, u64, p], i32),
            "aceapex_rans_status": ([p, p, ctypes.POINTER(u32)], i32),
            "aceapex_rans_static_setup": ([], i32),
            "aceapex_rans_encode_static": ([p, u64, u64, p, p, u64, p, p], i32),
            "aceapex_set_phase_timing": ([p, i32], i32),
            "aceapex_phase_times": ([p, ctypes.POINTER(ctypes.c_float)], i32),
        }
        for name, (args, res) in sig.items():
            f = getattr(L, name)
            f.argtypes, f.restype = args, res
        _lib = L
    return _lib


def _chk(rc, what=""):
    if rc:
        raise AceapexError(rc, what)


class Archive:
    """An archive resident in device memory.  `archive` is a uint8 numpy array / bytes (uploaded here) or a CUDA uint8
    torch tensor (used in place)."""

    def __init__(self, archive, device="cuda:0", stream=None):
        import torch
        self._torch = torch
        L = load()
        self.L = L
        if isinstance(archive, torch.Tensor) and archive.is_cuda:
            self.d_archive = archive
            host = None
        else:
            host = np.ascontiguousarray(np.frombuffer(archive, dtype=np.uint8) if isinstance(archive, (bytes, bytearray)) else archive)
            self.d_archive = torch.from_numpy(host).to(device)
        self.device = self.d_archive.device
        self.h = ctypes.c_void_p()
        with torch.cuda.device(self.device):
            _chk(L.aceapex_open(self.d_archive.data_ptr(), self.d_archive.numel(),
                                host.ctypes.data if host is not None else None, ctypes.byref(self.h)), "open")
        self._info = Info()
        _chk(L.aceapex_info(self.h, ctypes.byref(self._info)))
        self.workspace = torch.empty(max(int(self._info.workspace_bytes), 256), dtype=torch.uint8, device=self.device)
        _chk(L.aceapex_set_workspace(self.h, self.workspace.data_ptr(), self.workspace.numel()))
        if stream is not None:
            self.set_stream(stream)

    # -- plumbing
    def _chk(self, rc, what=""):
        if rc:
            raise AceapexError(rc, "%s (cuda error %d)" % (what, self.L.aceapex_last_cuda_error(self.h)) if rc == -8 else what)

    def info(self):
        return {k: int(getattr(self._info, k)) for k, _ in Info._fields_}

    @property
    def raw_bytes(self):
        return int(self._info.raw_bytes)

    def set_stream(self, stream):
        _chk(self.L.aceapex_set_stream(self.h, ctypes.c_void_p(stream.cuda_stream if stream is not None else 0)))

    def new_output(self, n=None):
        n = self.raw_bytes if n is None else n
        return self._torch.empty(max(n, 1), dtype=self._torch.uint8, device=self.device)

    def check(self):
        rc = self.L.aceapex_check(self.h)
        if rc:
            raise AceapexError(rc, "device flags 0x%x cuda %d" % (self.L.aceapex_device_flags(self.h),
                                                                   self.L.aceapex_last_cuda_error(self.h)))

    def set_phase_timing(self, on=True):
        _chk(self.L.aceapex_set_phase_timing(self.h, 1 if on else 0))

    def phase_times(self):
        """(literal launch, lower-level match launch, top-level match launch) of the last decode_all, in ms."""
        ms = (ctypes.c_float * 3)()
        _chk(self.L.aceapex_phase_times(self.h, ms), "phase_times")
        return [float(v) for v in ms]

    def launch_count(self):
        return int(self.L.aceapex_launch_count(self.h))

    def graph_launch_count(self):
        return int(self.L.aceapex_graph_launch_count(self.h))

    def close(self):
        if self.h:
            self.L.aceapex_close(self.h)
            self.h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the calls of include/aceapex.h
    def decode_all(self, out=None, levels=False, schedule=None):
        """schedule: None / "levels" (default: literal launch + one match launch per level), "flags" (two launches,
        completion flags) or "fused" (one launch)."""
        out = self.new_output() if out is None else out
        schedule = "levels" if levels else schedule
        f = {None: self.L.aceapex_decode_all, "levels": self.L.aceapex_decode_all, "flags": self.L.aceapex_decode_all_flags,
             "fused": self.L.aceapex_decode_all_fused}[schedule]
        self._chk(f(self.h, out.data_ptr()), "decode_all")
        return out[:self.raw_bytes]

    def decode_range(self, lo, hi, out=None, vram_budget=0):
        out = self.new_output(hi - lo) if out is None else out
        self._chk(self.L.aceapex_decode_range(self.h, lo, hi, out.data_ptr(), vram_budget), "decode_range")
        return out[:hi - lo]

    def reads_bytes(self, read_index, read_ids):
        total = ctypes.c_uint64()
        offs = np.zeros(len(read_ids) + 1, dtype=np.uint64)
        self._chk(self.L.aceapex_reads_bytes(read_index.ctypes.data, read_index.size, read_ids.ctypes.data, read_ids.size,
                                        ctypes.byref(total), offs.ctypes.data), "reads_bytes")
        return int(total.value), offs

    def decode_reads(self, read_index, read_ids, out=None):
        read_index = np.ascontiguousarray(read_index, dtype=np.uint64)
        read_ids = np.ascontiguousarray(read_ids, dtype=np.uint64)
        if out is None:
            total, _ = self.reads_bytes(read_index, read_ids)
            out = self.new_output(total)
        self._chk(self.L.aceapex_decode_reads(self.h, read_index.ctypes.data, read_index.size, read_ids.ctypes.data,
                                         read_ids.size, out.data_ptr()), "decode_reads")
        return out

    def decode_stream(self, lo, hi, ring, window_bytes, consumer=None, vram_budget=0):
        """Range decode through the ring tensor (aceapex_decode_stream).  consumer(window_index, lo, hi, d_window_ptr, stream_ptr)
        -> 0 to go on; None: the library's device FNV consumer.  Returns the statistics as a dict."""
        st = StreamStats()
        cb = WINDOW_FN(lambda user, w, a, b, ptr, stream: int(consumer(w, a, b, ptr, stream) or 0)) if consumer else WINDOW_FN()
        self._chk(self.L.aceapex_decode_stream(self.h, lo, hi, ring.data_ptr(), ring.numel(), window_bytes, cb, None, vram_budget,
                                               ctypes.byref(st)), "decode_stream")
        return {k: getattr(st, k) for k, _ in StreamStats._fields_ if k != "reserved"}

    def set_resident(self, slot, lo, hi, tensor):
        self._chk(self.L.aceapex_set_resident(self.h, slot, lo, hi, tensor.data_ptr() if tensor is not None else None))

    def verify_fnv(self, data, lo=0, hi=None):
        hi = self.raw_bytes if hi is None else hi
        bad = ctypes.c_uint64()
        self._chk(self.L.aceapex_verify_fnv(self.h, data.data_ptr(), lo, hi, ctypes.byref(bad)), "verify_fnv")
        return int(bad.value)

    def decode_all_host(self, h_archive, d_stage, h_out):
        """h_archive / h_out: pinned CPU uint8 tensors; d_stage: device uint8 tensor of raw_bytes."""
        self._chk(self.L.aceapex_decode_all_host(self.h, h_archive.data_ptr(), d_stage.data_ptr(), h_out.data_ptr()), "decode_all_host")


class RansBatch:
    """The entropy stage alone (include/aceapex.h, aceapex_rans_*): rows of byte symbols coded with one static
    table.  Marshalling only: tables, encode and decode run in the CUDA library."""

    def __init__(self, freq, row_bytes, device="cuda:0"):
        import torch
        self._torch, self.L, self.row_bytes = torch, load(), int(row_bytes)
        self.device = torch.device(device)
        self.stream = torch.cuda.current_stream(self.device)
        freq = np.ascontiguousarray(freq, dtype=np.uint16)
        self.row_cap = int(self.L.aceapex_rans_row_capacity(self.row_bytes))
        self.tables = torch.empty(int(self.L.aceapex_rans_table_bytes()), dtype=torch.uint8, device=self.device)
        with torch.cuda.device(self.device):
            self.scratch = torch.empty(int(self.L.aceapex_rans_scratch_bytes(self.row_bytes)), dtype=torch.uint8, device=self.device)
            _chk(self.L.aceapex_rans_tables(freq.ctypes.data, self.tables.data_ptr(), ctypes.c_void_p(self.stream.cuda_stream)), "rans_tables")

    def new_encoded(self, n_rows):
        t = self._torch
        return (t.empty(n_rows * self.row_cap + 128, dtype=t.uint8, device=self.device), t.empty(n_rows, dtype=t.int32, device=self.device))

    def encode(self, rows, enc=None, sizes=None):
        """rows: CUDA uint8 tensor (n_rows, row_bytes).  Returns (encoded buffer, int32 sizes per row); asynchronous."""
        n = rows.shape[0]
        if enc is None:
            enc, sizes = self.new_encoded(n)
        _chk(self.L.aceapex_rans_encode(rows.data_ptr(), n, self.row_bytes, self.tables.data_ptr(), enc.data_ptr(), self.row_cap, sizes.data_ptr(),
                                        self.scratch.data_ptr(), self.scratch.numel(), ctypes.c_void_p(self.stream.cuda_stream)), "rans_encode")
        return enc, sizes

    def encode_static(self, rows, enc=None, sizes=None):
        """encode() through aceapex_rans_encode_static: no scratch passed, nothing allocated by the library (row_bytes <= 65536)."""
        n = rows.shape[0]
        if enc is None:
            enc, sizes = self.new_encoded(n)
        with self._torch.cuda.device(self.device):
            _chk(self.L.aceapex_rans_encode_static(rows.data_ptr(), n, self.row_bytes, self.tables.data_ptr(), enc.data_ptr(), self.row_cap,
                                                   sizes.data_ptr(), ctypes.c_void_p(self.stream.cuda_stream)), "rans_encode_static")
        return enc, sizes

    def decode(self, enc, sizes, n_rows, out=None):
        t = self._torch
        out = t.empty((n_rows, self.row_bytes), dtype=t.uint8, device=self.device) if out is None else out
        _chk(self.L.aceapex_rans_decode(enc.data_ptr(), n_rows, self.row_bytes, self.row_cap, sizes.data_ptr(), self.tables.data_ptr(), out.data_ptr(),
                                        self.scratch.data_ptr(), self.scratch.numel(), ctypes.c_void_p(self.stream.cuda_stream)), "rans_decode")
        return out

    def status(self):
        v = ctypes.c_uint32()
        _chk(self.L.aceapex_rans_status(self.scratch.data_ptr(), ctypes.c_void_p(self.stream.cuda_stream), ctypes.byref(v)), "rans_status")
        return int(v.value)
