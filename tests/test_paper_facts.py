"""Pins against numbers the paper prints (tests/golden/paper_facts.txt): block-count arithmetic and units of the format,
the GB/s convention of the metric, the width of a read-index entry."""
import os
import struct
import sys

import numpy as np
import pytest

from oracle import acx_oracle as O

HERE = os.path.dirname(os.path.abspath(__file__))


def facts():
    out = {}
    for line in open(os.path.join(HERE, "golden", "paper_facts.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def header_only_archive(N, log2_bs, n_blocks, W):
    """A buffer that satisfies the header checks of FORMAT.md §1.1 (the oracle's header() reads nothing else)."""
    n_tables = 4 + W
    tables_off = 192
    qtab_off = tables_off + 528 * n_tables
    blocktab_off = qtab_off
    dir_off = (blocktab_off + 8 * (n_blocks + 1) + 15) // 16 * 16
    payload_off = dir_off + 32 * n_blocks
    total = payload_off + 128
    hdr = bytes([0x41, 0x43, 0x58, 0x42, 0x32, 0x30, 0x30, 0x00]) + struct.pack(
        "<IIQQQ" + "I" * 12 + "Q" * 13, 3, 192, N, n_blocks, n_blocks, log2_bs, 4, W, 11, n_tables, 0, 1, 0, min(log2_bs, 14), 0, 0, 0,
        tables_off, qtab_off, blocktab_off, dir_off, 0, payload_off, total, N, 0, 0, n_blocks, 0, 0)
    assert len(hdr) == 192
    return np.frombuffer(hdr, dtype=np.uint8), total


def header_fields(N, log2_bs, n_blocks, W):
    """The oracle's view of that header (the sections it describes are never touched: 3 M blocks would be 120 MB)."""
    hdr, total = header_only_archive(N, log2_bs, n_blocks, W)
    import ctypes
    f = np.zeros(len(O.HEADER_FIELDS), dtype=np.uint64)
    rc = O._load().acx_oracle_header(hdr.ctypes.data, total, f.ctypes.data)     # archive_bytes = what the header claims
    if rc:
        raise O.OracleError(rc)
    return {k: int(v) for k, v in zip(O.HEADER_FIELDS, f)}


def test_block_count_of_the_papers_50GB_file():
    f = facts()
    N, bs = int(f["output_bytes_50GB"]), int(f["block_size_16KB"])
    assert bs == 1 << 14
    want = int(f["blocks_of_50GB_at_16KB"])
    assert -(-N // bs) == want                       # ceil(N / BS) with 16 KB = 16,384 B and GB = 10^9 B
    h = header_fields(N, 14, want, 5)                 # 50e9 needs 36 bits: W = 5 offset bytes
    assert h["n_blocks"] == want and h["N"] == N
    for wrong in (want - 1, want + 1):
        with pytest.raises(O.OracleError):
            header_fields(N, 14, wrong, 5)
    with pytest.raises(O.OracleError):               # 4 offset bytes cannot address 50 GB (the uint32 overflow)
        header_fields(N, 14, want, 4)


def test_throughput_convention():
    f = facts()
    sys.path.insert(0, os.path.dirname(HERE))
    import bench
    got = bench.aggregate_value(1, f["output_bytes_50GB"], f["range_decode_ms_50GB"])
    assert abs(got - f["range_decode_GBps_50GB"]) < 0.06      # 50e9 B / 301.7 ms = 165.73 GB/s


def test_index_entry_is_8_bytes_per_read():
    f = facts()
    from paper_2606_18900_b200 import datagen
    idx = datagen.fastq_index(1 << 20)
    assert idx.dtype == np.uint64 and idx.itemsize * int(f["index_reads"]) == int(f["index_bytes"])
    # FORMAT.md §4: offset in bits 0..39, length in bits 40..63; the block of a read is offset >> log2(block size)
    off = idx & np.uint64((1 << 40) - 1)
    ln = idx >> np.uint64(40)
    assert int(off[0]) == 0 and (np.diff(off.astype(np.int64)) == ln[:-1].astype(np.int64)).all()
