"""Parity of the CUDA path (through the C ABI, include/aceapex.h) with the oracle and the original bytes."""
import numpy as np
import pytest
import torch

from acx_build import build
from oracle import acx_oracle as O

pytestmark = pytest.mark.gpu


def gpu_decode(archive, levels=False, schedule=None):
    from paper_2606_18900_b200.aceapex import Archive
    ar = Archive(archive)
    out = ar.decode_all(levels=levels, schedule=schedule)
    ar.check()
    res = out.cpu().numpy().copy()
    ar.close()
    return res


HAND = [
    ([[(b"hello", None)]], 5, 3, {}),
    ([[(b"a", (0, 7))], [(b"", (0, 8))], [(b"", (8, 8))], [(b"", (16, 3))]], 27, 3, dict(min_match=3, levels=[0, 1, 2, 3])),
    ([[(b"abc", (0, 10))]], 13, 4, {}),
    ([[(b"wxyz", (0, 4))]], 8, 3, {}),
    ([[(b"abcd", (0, 4))], [(b"", (2, 5)), (b"XYZ", None)]], 16, 3, dict(levels=[0, 1])),
    ([[(b"01234567", None)], [(b"89ab", (6, 4))], [(b"", (6, 5)), (b"!!!", None)]], 24, 3, {}),
    ([[(b"ACGTACGT", None)], [(b"", (0, 4)), (b"", (4, 4))]], 16, 3, {}),
    ([[(b"ABCDEFGH", None)], [(b"", (0, 8))], [(b"", (8, 8))]], 24, 3, dict(levels=[0, 0, 1])),
    ([[(b"xy", (0, 9)), (b"END", None)]], 14, 4, {}),
]


# version 3 of the format: segments, literal classes, pair symbols (the archives of tests/test_oracle_handbuilt.py)
SEGS3 = [[(b"ABCDEFGHIJ", None)], [(b"KL", (0, 3)), (b"mn", (2, 4))], [(b"", (8, 4)), (b"wxyz123", None)]]
QCMDS = [(b"ab", (0, 2)), (b"QQQQQ", (4, 3)), (b"XY", (4, 4)), (b"RSTUVW", (12, 2)), (b"!", None)]
QFIRST = [(b"a" + bytes(range(98, 98 + 30)) + b"~", None)]
QPAIR = [QFIRST, [(b"p", (0, 2)), (b"HIJKL", (35, 2)), (b"MNOPQ", (0, 2)), (b"xyzw", None)]]
HAND += [
    ([SEGS3], 32, 5, dict(log2_seg=3, min_match=2)),
    ([SEGS3, [(b"", (0, 8))]], 40, 5, dict(log2_seg=3, min_match=2)),
    ([QCMDS], 27, 5, dict(min_match=2, q_min=4)),
    ([QCMDS], 27, 5, dict(min_match=2, q_min=4, q_mode=1)),
    ([QCMDS], 27, 5, dict(min_match=2, q_min=2, q_mode=1)),
    (QPAIR, 53, 5, dict(min_match=2, q_min=4, q_mode=1)),
    (QPAIR, 53, 5, dict(min_match=2, q_min=4, q_mode=1, filler=0)),
    (QPAIR, 53, 5, dict(min_match=2, q_min=4, q_mode=0)),
    ([[[(b"ab", None)], [(b"ab", (2, 4))]]], 8, 3, dict(min_match=2)),
    ([[(b"xab", (1, 5))]], 8, 3, dict(min_match=2)),
]


@pytest.mark.parametrize("case", range(len(HAND)))
@pytest.mark.parametrize("levels", [False, True])
def test_hand_built(case, levels):
    blocks, N, lb, kw = HAND[case]
    a = build(blocks, N, lb, **kw)
    exp = O.decode(a)
    got = gpu_decode(a, schedule="flags" if levels else None)
    assert got.tobytes() == exp.tobytes()
    if not levels:
        assert gpu_decode(a, schedule="fused").tobytes() == exp.tobytes()


def test_hand_built_escapes_and_planes():
    lit = bytes((i * 7 + 3) % 251 for i in range(300))
    blocks = [[(lit, (0, 300)), (b"", (10, 4 + 255)), (lit[:255], (1, 4 + 254)), (b"q", None)]]
    N = 300 + 300 + 259 + 255 + 258 + 1
    for raw in [(), (0,), (0, 1), (0, 1, 2, 3)]:
        a = build(blocks, N, 11, raw_planes=raw)
        assert gpu_decode(a).tobytes() == O.decode(a).tobytes()


@pytest.mark.parametrize("schedule", [None, "flags", "fused"])
def test_config0_fastq(fastq_4m, fastq_4m_archive, schedule):
    got = gpu_decode(fastq_4m_archive, schedule=schedule)
    assert np.array_equal(got, O.decode(fastq_4m_archive))      # bit-exact vs the oracle
    assert np.array_equal(got, fastq_4m)                         # and vs the original bytes


def test_fasta(fasta_2m, fasta_2m_archive):
    got = gpu_decode(fasta_2m_archive)
    assert np.array_equal(got, fasta_2m)


@pytest.mark.parametrize("kw", [dict(q_mode=0), dict(q_mode=1), dict(q_min=0), dict(q_min=2), dict(q_min=2, q_mode=0), dict(q_min=300, q_mode=1),
                                dict(max_level=3), dict(max_level=3, q_mode=0), dict(block_size=65536, log2_seg=12), dict(block_size=4096, log2_seg=9),
                                dict(block_size=1 << 18, q_mode=0, max_level=2), dict(block_size=1 << 20, max_level=1)])
def test_encoder_options_of_version_3(fastq_4m, fasta_2m, kw):
    """Literal classes, pair symbols, segment sizes and level caps (FORMAT.md 1.5-1.7, 3), every schedule, vs the oracle."""
    from paper_2606_18900_b200 import encoder
    for x in (fastq_4m[:(2 << 20) + 4321], fasta_2m[:(1 << 20) + 77]):
        a = encoder.encode(x, **kw)
        exp = O.decode(a)
        assert np.array_equal(exp, x)
        for sched in (None, "flags", "fused"):
            assert np.array_equal(gpu_decode(a, schedule=sched), exp), (kw, sched)


def test_incompressible_and_huge_runs():
    """Literal runs and matches longer than a segment: runs cut at segment boundaries, one command of 200,000 match bytes."""
    from paper_2606_18900_b200 import encoder
    rng = np.random.default_rng(5)
    noise = rng.integers(0, 256, 100_000, dtype=np.uint8)
    x = np.concatenate([noise, np.full(200_000, 65, np.uint8), noise[:50_000], np.tile(noise[:3000], 30)])
    for bs in (1 << 20, 1 << 16, 1 << 14):
        a = encoder.encode(x, block_size=bs)
        for sched in (None, "flags", "fused"):
            assert np.array_equal(gpu_decode(a, schedule=sched), x), (bs, sched)


@pytest.mark.parametrize("bs", [4096, 8192, 65536, 262144, 1 << 20])
def test_block_sizes(fastq_4m, bs):
    from paper_2606_18900_b200 import encoder
    x = fastq_4m[:(3 << 20) + 12345]            # ragged tail
    a = encoder.encode(x, block_size=bs)
    assert np.array_equal(gpu_decode(a), x)
    assert np.array_equal(gpu_decode(a, schedule="flags"), x)
    assert np.array_equal(gpu_decode(a, schedule="fused"), x)


def test_runs_and_periods():
    from paper_2606_18900_b200 import encoder
    for data in (b"N" * 100000, (b"ACGTTGCA" * 7 + b"\n") * 3000, b"x" + b"\0" * 70000 + b"y", b"", b"q"):
        x = np.frombuffer(data, dtype=np.uint8)
        a = encoder.encode(x, block_size=4096)
        assert gpu_decode(a).tobytes()[:len(data)] == data


def test_repeated_calls_and_fnv(fastq_4m, fastq_4m_archive):
    from paper_2606_18900_b200.aceapex import Archive
    ar = Archive(fastq_4m_archive)
    out = ar.new_output()
    for _ in range(3):
        out.zero_()
        ar.decode_all(out)
        ar.check()
        assert ar.verify_fnv(out) == 0
    out[12345] ^= 1
    assert ar.verify_fnv(out) == 1
    assert torch.equal(out.cpu()[:12345], torch.from_numpy(fastq_4m[:12345]))
    ar.close()


def test_flag_schedules_stress(fastq_4m, monkeypatch):
    """The completion-count protocol (S20) under repetition: compute-sanitizer is refused on this GPU pool, so the
    flag-driven schedules are run 200 times per CTA size on configs[0] encoded with a deep level structure (max_level 7: most
    blocks wait for others), every output compared with the original bytes on the device; then flag-driven windows."""
    from paper_2606_18900_b200 import encoder
    from paper_2606_18900_b200.aceapex import Archive
    a = encoder.encode(fastq_4m, block_size=16384, max_level=7)
    want = torch.from_numpy(fastq_4m).cuda()
    rng = np.random.default_rng(8)
    for threads in ("1024", "512", "192"):
        monkeypatch.setenv("ACEAPEX_THREADS", threads)
        ar = Archive(a)
        monkeypatch.delenv("ACEAPEX_THREADS")
        assert ar.info()["max_level"] >= 5
        out = ar.new_output()
        for k in range(200):
            sched = ("flags", "fused", None)[k % 3]
            out.fill_(0xA5)
            ar.decode_all(out, schedule=sched)
            assert torch.equal(out[:want.numel()], want), (threads, k, sched)
        ar.check()
        buf = ar.new_output(1 << 20)
        for k in range(60):                                      # windows of 3..60 blocks: flag-driven, in index order
            lo = int(rng.integers(0, 190)) * 16384
            hi = lo + int(rng.integers(3, 60)) * 16384
            buf.fill_(0x5A)
            ar.decode_range(lo, hi, out=buf)
            assert torch.equal(buf[:hi - lo], want[lo:hi]), (threads, lo, hi)
        ar.check()
        ar.close()


def test_open_errors(fastq_4m_archive):
    from paper_2606_18900_b200.aceapex import AceapexError, Archive
    bad = fastq_4m_archive.copy()
    bad[0] = 0
    with pytest.raises(AceapexError) as e:
        Archive(bad)
    assert e.value.name == "E_MAGIC"
    with pytest.raises(AceapexError) as e:
        Archive(fastq_4m_archive[:-4096].copy())
    assert e.value.name == "E_TRUNCATED"
    bad = fastq_4m_archive.copy()
    h = O.header(fastq_4m_archive)
    bad[h["dir_off"] + 16:h["dir_off"] + 18] = 0         # n_cmd = 0
    with pytest.raises(AceapexError) as e:
        Archive(bad)
    assert e.value.name == "E_CORRUPT"


def test_device_integrity_flag(fastq_4m_archive):
    from paper_2606_18900_b200.aceapex import AceapexError, Archive
    bad = fastq_4m_archive.copy()
    h = O.header(fastq_4m_archive)
    bad[h["payload_off"] + 200] ^= 0x55                  # inside block 0's word stream
    ar = Archive(bad)
    ar.decode_all()
    with pytest.raises(AceapexError) as e:
        ar.check()
    assert e.value.name == "E_CORRUPT"
    ar.close()


def test_wide_offsets_many_coded_planes_fewer_warps_per_cta():
    """W = 8 with every offset plane rANS-coded: 11 decode tables (88 KB) leave room for fewer than 32 warps per CTA, so
    the library launches smaller CTAs; every schedule, a range and reads must still be exact."""
    from paper_2606_18900_b200.aceapex import Archive
    lit = bytes((i * 7 + 3) % 251 for i in range(300))
    blocks = [[(lit, (0, 300)), (b"", (10, 4 + 255)), (lit[:255], (1, 4 + 254)), (b"q", None)]]
    N = 300 + 300 + 259 + 255 + 258 + 1
    for W, raw in ((8, ()), (8, (0, 3, 7)), (6, ()), (5, (0,))):
        a = build(blocks, N, 11, W=W, raw_planes=raw)
        exp = O.decode(a).tobytes()
        for sched in (None, "flags", "fused"):
            assert gpu_decode(a, schedule=sched).tobytes() == exp, (W, raw, sched)
        ar = Archive(a)
        assert ar.decode_range(100, 1200).cpu().numpy().tobytes() == exp[100:1200]
        idx = np.array([(5 | (700 << 40)), (900 | (300 << 40))], dtype=np.uint64)
        got = ar.decode_reads(idx, np.array([1, 0, 1], dtype=np.uint64)).cpu().numpy().tobytes()
        assert got[:1300] == exp[900:1200] + exp[5:705] + exp[900:1200]
        ar.check()
        ar.close()


def test_output_must_be_16_byte_aligned(fastq_4m_archive):
    from paper_2606_18900_b200.aceapex import AceapexError, Archive
    ar = Archive(fastq_4m_archive)
    out = ar.new_output(ar.raw_bytes + 64)
    with pytest.raises(AceapexError) as e:
        ar.decode_all(out[8:])
    assert e.value.name == "E_ARG"
    ar.close()


def test_phase_times(fastq_4m_archive):
    from paper_2606_18900_b200.aceapex import AceapexError, Archive
    ar = Archive(fastq_4m_archive)
    with pytest.raises(AceapexError):
        ar.phase_times()                                     # timing is off
    ar.set_phase_timing(True)
    out = ar.decode_all()
    ms = ar.phase_times()
    ar.check()
    assert len(ms) == 3 and ms[0] > 0 and ms[2] > 0 and all(v >= 0 for v in ms)
    ar.set_phase_timing(False)
    ar.close()
