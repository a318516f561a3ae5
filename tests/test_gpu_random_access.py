"""decode_range / decode_reads (§4): bit-exact against slices of the ORIGINAL bytes and against the
oracle's whole-file output."""
import numpy as np
import pytest
import torch

from acx_build import build
from oracle import acx_oracle as O

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fq(fastq_4m, fastq_4m_archive):
    from paper_2606_18900_b200.aceapex import Archive
    ar = Archive(fastq_4m_archive)
    yield ar, fastq_4m
    ar.close()


@pytest.fixture(scope="module")
def fa(fasta_2m, fasta_2m_archive):
    from paper_2606_18900_b200.aceapex import Archive
    ar = Archive(fasta_2m_archive)
    yield ar, fasta_2m
    ar.close()


def check_range(ar, x, lo, hi):
    got = ar.decode_range(lo, hi)
    ar.check()
    assert got.cpu().numpy().tobytes() == x[lo:hi].tobytes(), (lo, hi)


def test_ranges_fastq(fq):
    ar, x = fq
    N = x.size
    rng = np.random.default_rng(0)
    cases = [(0, 0), (5, 5), (0, 1), (N - 1, N), (0, N), (16384, 32768), (16383, 16385), (100, 200), (1, N - 1),
             (N - 40000, N), (3 * 16384, 3 * 16384 + 1), (16384 * 100 + 7, 16384 * 101 - 9)]
    for _ in range(12):
        lo = int(rng.integers(0, N))
        hi = int(min(N, lo + rng.integers(0, 400000)))
        cases.append((lo, hi))
    for lo, hi in cases:
        check_range(ar, x, lo, hi)


def test_ranges_far_from_start_need_sources_before_lo(fq):
    ar, x = fq
    N = x.size
    # the last quarter of the file reads from everywhere before it
    check_range(ar, x, 3 * N // 4 + 123, N - 77)
    check_range(ar, x, N // 2, N // 2 + 5 * 16384)


def test_ranges_fasta(fa):
    ar, x = fa
    N = x.size
    rng = np.random.default_rng(1)
    for _ in range(10):
        lo = int(rng.integers(0, N))
        hi = int(min(N, lo + rng.integers(1, 300000)))
        check_range(ar, x, lo, hi)
    check_range(ar, x, 0, N)


def test_range_errors(fq):
    from paper_2606_18900_b200.aceapex import AceapexError
    ar, x = fq
    with pytest.raises(AceapexError) as e:
        ar.decode_range(10, 5)
    assert e.value.name == "E_RANGE"
    with pytest.raises(AceapexError) as e:
        ar.decode_range(0, x.size + 1)
    assert e.value.name == "E_RANGE"
    with pytest.raises(AceapexError) as e:
        ar.decode_range(0, 100, vram_budget=4096)
    assert e.value.name == "E_BUDGET"


def test_reads_fastq(fq):
    from paper_2606_18900_b200 import datagen
    ar, x = fq
    idx = datagen.fastq_index(x.size)
    rng = np.random.default_rng(2)
    for n in (1, 2, 33, 4096):
        ids = rng.integers(0, idx.size, n).astype(np.uint64)
        ids[-1] = ids[0]                                # a duplicate
        total, offs = ar.reads_bytes(idx, ids)
        got = ar.decode_reads(idx, ids).cpu().numpy()
        ar.check()
        for k, r in enumerate(ids):
            o, ln = int(idx[r] & np.uint64((1 << 40) - 1)), int(idx[r] >> np.uint64(40))
            assert got[int(offs[k]):int(offs[k]) + ln].tobytes() == x[o:o + ln].tobytes()
        assert total == int(offs[-1])
    # first and last read, and a read that crosses a block boundary
    off = (idx & np.uint64((1 << 40) - 1)).astype(np.int64)
    ln = (idx >> np.uint64(40)).astype(np.int64)
    crossing = np.nonzero((off >> 14) != ((off + ln - 1) >> 14))[0][:5]
    ids = np.concatenate([[0, idx.size - 1], crossing]).astype(np.uint64)
    got = ar.decode_reads(idx, ids).cpu().numpy()
    exp = np.concatenate([x[off[i]:off[i] + ln[i]] for i in ids.astype(np.int64)])
    assert got[:exp.size].tobytes() == exp.tobytes()


def test_single_reads_one_cta_many_warps():
    """A single read goes through k_spans_cta (one CTA, a shared queue of spans, many warps): 400 single reads on FASTQ and
    FASTA archives with 0, 2 and 7 dependency levels, long reads (32 KB, several segments) included, vs the original bytes."""
    from paper_2606_18900_b200 import datagen, encoder
    from paper_2606_18900_b200.aceapex import Archive
    rng = np.random.default_rng(12)
    for x in (datagen.fastq(7, 3 << 20, 1_000_000), datagen.fasta(8, 2 << 20)):
        for ml in (0, 2, 7):
            ar = Archive(encoder.encode(x, block_size=16384, max_level=ml))
            offs = rng.integers(0, x.size - 40_000, 400).astype(np.uint64)
            lens = np.where(np.arange(400) % 50 == 0, 32_768, rng.integers(1, 700, 400)).astype(np.uint64)
            idx = offs | (lens << np.uint64(40))
            out = ar.new_output(40_000)
            for i in range(400):
                ar.decode_reads(idx, np.array([i], dtype=np.uint64), out=out)
                o, ln = int(offs[i]), int(lens[i])
                assert out[:ln].cpu().numpy().tobytes() == x[o:o + ln].tobytes(), (ml, i, o, ln)
            ar.check()
            ar.close()


def test_reads_regions_fasta(fa):
    from paper_2606_18900_b200 import datagen
    ar, x = fa
    idx = datagen.region_index(3, x.size, 5000, 150)
    ids = np.arange(5000, dtype=np.uint64)
    got = ar.decode_reads(idx, ids).cpu().numpy()
    ar.check()
    off = (idx & np.uint64((1 << 40) - 1)).astype(np.int64)
    exp = np.concatenate([x[o:o + 150] for o in off])
    assert got[:exp.size].tobytes() == exp.tobytes()


def test_reads_errors(fq):
    from paper_2606_18900_b200 import datagen
    from paper_2606_18900_b200.aceapex import AceapexError
    ar, x = fq
    idx = datagen.fastq_index(x.size)
    with pytest.raises(AceapexError) as e:
        ar.decode_reads(idx, np.array([idx.size], dtype=np.uint64))
    assert e.value.name == "E_RANGE"


def test_resident_window_serves_as_source(fq):
    """PAPER.md:107-109 §5: consecutive windows through a ring; an earlier window stays resident as a match source."""
    ar, x = fq
    W = 64 * 16384
    ring = [ar.new_output(W) for _ in range(2)]
    for w in range(x.size // W):
        buf = ring[w % 2]
        ar.set_resident(w % 2, 0, 0, None)          # this buffer is about to be overwritten: no longer a source
        got = ar.decode_range(w * W, (w + 1) * W, out=buf)
        ar.check()
        assert torch.equal(got.cpu(), torch.from_numpy(x[w * W:(w + 1) * W]))
        ar.set_resident(w % 2, w * W, (w + 1) * W, buf)
    ar.set_resident(0, 0, 0, None)
    ar.set_resident(1, 0, 0, None)


HAND = [
    ([[(b"a", (0, 7))], [(b"", (0, 8))], [(b"", (8, 8))], [(b"", (16, 3))]], 27, 3, dict(min_match=3, levels=[0, 1, 2, 3])),
    ([[(b"abc", (0, 10)), (b"XYZ", None)], [(b"", (1, 9)), (b"0123456", None)]], 32, 4, dict(levels=[0, 1])),
    ([[(b"01234567", None)], [(b"89ab", (6, 4))], [(b"", (6, 5)), (b"!!!", None)]], 24, 3, {}),
    ([[(b"ABCDEFGH", None)], [(b"", (0, 8))], [(b"", (8, 8))]], 24, 3, dict(levels=[0, 0, 1])),
    ([[[(b"ABCDEFGHIJ", None)], [(b"KL", (0, 3)), (b"mn", (2, 4))], [(b"", (8, 4)), (b"wxyz123", None)]], [(b"", (0, 8))]], 40, 5,
     dict(log2_seg=3, min_match=2)),
    ([[(b"a" + bytes(range(98, 98 + 30)) + b"~", None)], [(b"p", (0, 2)), (b"HIJKL", (35, 2)), (b"MNOPQ", (0, 2)), (b"xyzw", None)]], 53, 5,
     dict(min_match=2, q_min=4, q_mode=1)),
    ([[(b"a" + bytes(range(98, 98 + 30)) + b"~", None)], [(b"p", (0, 2)), (b"HIJKL", (35, 2)), (b"MNOPQ", (0, 2)), (b"xyzw", None)]], 53, 5,
     dict(min_match=2, q_min=4, q_mode=0)),
]


@pytest.mark.parametrize("case", range(len(HAND)))
def test_hand_built_every_range(case):
    from paper_2606_18900_b200.aceapex import Archive
    blocks, N, lb, kw = HAND[case]
    a = build(blocks, N, lb, **kw)
    exp = O.decode(a).tobytes()
    ar = Archive(a)
    for lo in range(0, N + 1):
        for hi in range(lo, N + 1, 3):
            got = ar.decode_range(lo, hi).cpu().numpy().tobytes()[:hi - lo]
            assert got == exp[lo:hi], (lo, hi)
    ar.check()
    ar.close()


@pytest.fixture(scope="module")
def big(request):
    """12 MiB FASTQ (high coverage: most matches reach far back) and 8 MiB FASTA: windows of >= 256 blocks take the
    aggregated-demand path of decode_range (literals, demand rounds, matches per level)."""
    from paper_2606_18900_b200 import datagen, encoder
    from paper_2606_18900_b200.aceapex import Archive
    xq = datagen.fastq(7, 12 << 20, 300_000)
    xa = datagen.fasta(9, 8 << 20)
    aq, aa = Archive(encoder.encode(xq, block_size=16384)), Archive(encoder.encode(xa, block_size=16384))
    yield (aq, xq), (aa, xa)
    aq.close()
    aa.close()


def test_large_windows_with_foreign_sources(big):
    for ar, x in big:
        N = x.size
        BS = 16384
        for lo, hi in ((150 * BS, 450 * BS), (N - 300 * BS - 5, N), (100 * BS + 77, 400 * BS + 99), (0, 256 * BS), (5, N - 5),
                       (N // 3 - 3, N // 3 + 200 + 257 * BS)):
            check_range(ar, x, lo, min(hi, N))


@pytest.mark.parametrize("kw", [dict(max_level=3), dict(max_level=2, q_mode=0), dict(block_size=1 << 20, max_level=3), dict(block_size=65536),
                                dict(block_size=4096, q_min=0), dict(block_size=1 << 18, log2_seg=12, max_level=1)])
def test_large_windows_levels_and_segments(kw):
    """Archives with dependency levels (demand rounds recurse, the window's match launch is flag-driven) and with several
    segments per block: windows, ragged ends, reads; also a window placed at an ODD device address (pair stores fall back
    to byte stores)."""
    from paper_2606_18900_b200 import datagen, encoder
    from paper_2606_18900_b200.aceapex import Archive
    x = datagen.fastq(7, 6 << 20, 300_000)
    ar = Archive(encoder.encode(x, **kw))
    for lo, hi in ((100 * 16384, 380 * 16384), (x.size - 300 * 16384 - 5, x.size), (0, 256 * 16384), (1 << 20, (1 << 20) + 1), (3_000_001, 5_500_003)):
        check_range(ar, x, lo, hi)
    buf = ar.new_output((2 << 20) + 64)
    for shift in (1, 3, 8):
        lo, hi = (2 << 20) + 5, (4 << 20) + 5
        got = ar.decode_range(lo, hi, out=buf[shift:])
        ar.check()
        assert got.cpu().numpy().tobytes() == x[lo:hi].tobytes(), shift
    idx = datagen.fastq_index(x.size)
    rng = np.random.default_rng(3)
    off, ln = (idx & np.uint64((1 << 40) - 1)).astype(np.int64), (idx >> np.uint64(40)).astype(np.int64)
    for n in (1, 40, 3000):
        ids = rng.integers(0, idx.size, n).astype(np.uint64)
        got = ar.decode_reads(idx, ids).cpu().numpy()
        ar.check()
        _, offs = ar.reads_bytes(idx, ids)
        for k in range(0, n, 7):
            r = int(ids[k])
            assert got[int(offs[k]):int(offs[k]) + ln[r]].tobytes() == x[off[r]:off[r] + ln[r]].tobytes(), (n, k)
    ar.close()


def test_large_windows_ring(big):
    """Consecutive 4 MiB windows through a two-slot ring: sources are found in the window, in the resident previous
    window, or are reconstructed through the demand lists."""
    for ar, x in big:
        W = 256 * 16384
        ring = [ar.new_output(W) for _ in range(2)]
        for w in range((x.size + W - 1) // W):
            lo, hi = w * W, min(x.size, (w + 1) * W)
            buf = ring[w % 2]
            ar.set_resident(w % 2, 0, 0, None)
            got = ar.decode_range(lo, hi, out=buf)
            ar.check()
            assert torch.equal(got.cpu(), torch.from_numpy(x[lo:hi])), w
            ar.set_resident(w % 2, lo, hi, buf)
        ar.set_resident(0, 0, 0, None)
        ar.set_resident(1, 0, 0, None)


def test_large_window_runs_and_overlaps():
    """RLE runs and short periods that cross block and window boundaries (self-overlapping matches whose seed lies
    outside the window)."""
    from paper_2606_18900_b200 import encoder
    from paper_2606_18900_b200.aceapex import Archive
    rng = np.random.default_rng(3)
    parts = []
    for k in range(120):
        parts.append(rng.integers(65, 70, 3000 + 17 * k, dtype=np.uint8).tobytes())
        parts.append(b"N" * (20000 + 999 * (k % 7)))
        parts.append((b"ACGTTGCA" * 5 + b"\n") * 300)
    x = np.frombuffer(b"".join(parts), dtype=np.uint8)
    ar = Archive(encoder.encode(x, block_size=4096))
    N = x.size
    for lo, hi in ((300 * 4096, 700 * 4096), (N // 3 + 11, N // 3 + 11 + 300 * 4096), (N - 260 * 4096, N)):
        check_range(ar, x, lo, hi)
    ar.close()


def test_hot_source_segment_and_long_period_overlaps_through_the_demand_rounds():
    """One early segment (an N-run with newlines: self-overlapping matches of period 61) is the source of thousands of later
    matches, some of them kilobytes long: windows far from it get its bytes through the demand rounds (records of at most
    96 bytes, work items of 128 records, seeds copied piecewise), single reads through the per-warp recursion.  Every
    level cap, vs the original bytes and the oracle."""
    from paper_2606_18900_b200 import encoder
    from paper_2606_18900_b200.aceapex import Archive
    rng = np.random.default_rng(9)
    nrun = (b"N" * 60 + b"\n") * 400                         # 24,400 bytes, period 61
    odd = (b"ACGTTGCAGGA" * 7 + b"\n") * 200                 # period 78
    parts = [b">chr1\n", rng.integers(65, 69, 40_000, dtype=np.uint8).tobytes(), nrun, odd]
    for k in range(1500):
        parts.append(rng.integers(65, 69, 700 + (k % 13), dtype=np.uint8).tobytes())
        cut = 61 * (k % 300) + (k % 61)
        parts.append(nrun[cut:cut + 30 + (k * 37) % 3000])    # pieces of the run, 30 bytes .. 3 KB
        if k % 5 == 0:
            parts.append(odd[(k * 7) % 500:(k * 7) % 500 + 200 + k % 900])
    x = np.frombuffer(b"".join(parts), dtype=np.uint8)
    N = x.size
    for ml in (0, 1, 2):
        a = encoder.encode(x, block_size=16384, max_level=ml)
        want = O.decode(a)
        assert np.array_equal(want, x)
        ar = Archive(a)
        for lo, hi in ((N // 2, N // 2 + (1 << 20)), (N - (1 << 20) - 12345, N - 7), (N // 3 + 5, N // 3 + 5 + 70_000)):
            check_range(ar, x, lo, hi)
        idx = np.array([(N // 2 + 1000 * i) | (1500 << 40) for i in range(600)], dtype=np.uint64)
        for ids in (np.array([17], dtype=np.uint64), np.arange(600, dtype=np.uint64)):
            got = ar.decode_reads(idx, ids).cpu().numpy()
            ar.check()
            for j, i in enumerate(ids.tolist()):
                off = N // 2 + 1000 * i
                assert got[1500 * j:1500 * (j + 1)].tobytes() == x[off:off + 1500].tobytes(), (ml, i)
        ar.close()


def test_seeks_replayed_as_cuda_graphs_match_plain_launches(monkeypatch):
    """aceapex_decode_range of up to 8 MiB replays its launch sequence as a CUDA graph with updated node parameters
    (aceapex_graph_launch_count counts the replays); ACEAPEX_NO_GRAPHS=1 at open keeps the plain launches.  Both against
    the original bytes, for an archive without levels and for the encoder's default (flag-driven window launch)."""
    from paper_2606_18900_b200 import datagen, encoder
    from paper_2606_18900_b200.aceapex import Archive
    x = datagen.fastq(5, 6 << 20, 1_000_000)
    rng = np.random.default_rng(4)
    for kw in (dict(max_level=0), dict(), dict(block_size=65536, max_level=3)):
        a = encoder.encode(x, **kw)
        ar_g = Archive(a)
        monkeypatch.setenv("ACEAPEX_NO_GRAPHS", "1")
        ar_p = Archive(a)
        monkeypatch.delenv("ACEAPEX_NO_GRAPHS")
        BS = ar_g.info()["block_size"]
        n_calls = 0
        for k in range(40):
            blocks = (1, 3, 100 if BS == 16384 else 20)[k % 3]
            lo = int(rng.integers(0, x.size // BS - blocks)) * BS + (0 if k % 4 else 777)      # aligned and ragged
            hi = min(x.size, lo + blocks * BS - (0 if k % 5 else 13))
            want = x[lo:hi].tobytes()
            assert ar_g.decode_range(lo, hi).cpu().numpy().tobytes() == want, (kw, lo, hi)
            assert ar_p.decode_range(lo, hi).cpu().numpy().tobytes() == want, (kw, lo, hi)
            n_calls += 1
        ar_g.check(); ar_p.check()
        assert ar_g.graph_launch_count() == n_calls and ar_p.graph_launch_count() == 0, kw
        ar_g.close(); ar_p.close()


def test_end_to_end_host_pipeline(big, fq):
    """aceapex_decode_all_host: archive from pinned host memory, output to pinned host memory, chunks pipelined."""
    for ar, x in (big[0], big[1], fq):
        import torch as T
        h_arch = ar.d_archive.cpu().pin_memory()
        ar.d_archive.zero_()                                  # the call must bring every archive byte itself
        stage = ar.new_output()
        h_out = T.empty(x.size, dtype=T.uint8).pin_memory()
        for _ in range(2):
            h_out.zero_()
            ar.decode_all_host(h_arch, stage, h_out)
            ar.check()
            assert T.equal(h_out, T.from_numpy(x))


def test_small_vram_budget_means_more_sub_windows_not_failure(big):
    """vram_budget below the full workspace shrinks the demand lists: the window is served in several sub-windows."""
    from paper_2606_18900_b200.aceapex import AceapexError
    ar, x = big[0]
    need = ar.info()["workspace_bytes"]
    lo, hi = 200 * 16384, 700 * 16384
    served = 0
    for budget in (need - 1, need - (1 << 20), need - (4 << 20), need - (7 << 20), need // 2):
        try:
            got = ar.decode_range(lo, hi, vram_budget=budget)
        except AceapexError as e:
            assert e.name == "E_BUDGET"                      # below the floor: refused, never wrong
            continue
        ar.check()
        assert got.cpu().numpy().tobytes() == x[lo:hi].tobytes(), budget
        served += 1
    assert served >= 3


def test_decode_stream_ring_in_the_library(big):
    """aceapex_decode_stream: the library owns window order, slot rotation and resident registration.  A
    file larger than the ring, (a) checked by the library's own device FNV consumer, (b) handed window by window to a
    consumer that only counts callbacks and compares each window with the original bytes, (c) stopped by the consumer."""
    import ctypes
    from paper_2606_18900_b200.aceapex import AceapexError
    for ar, x in big:
        N = x.size
        W = 64 * 16384                                    # 1 MiB windows
        ring = ar.new_output(3 * W + 4096)                # three slots (and some slack the library must not need)
        st = ar.decode_stream(0, N, ring, W)
        assert st["n_windows"] == (N + W - 1) // W and st["n_slots"] == 3 and st["bytes"] == N and st["bad_blocks"] == 0
        assert st["device_ms"] > 0 and 0 < st["min_window_gbs"] <= st["max_window_gbs"]
        assert st["peak_device_bytes"] == ar.info()["archive_bytes"] + 3 * W + ar.info()["workspace_bytes"]
        seen = []

        errors0 = []

        def consumer(w, lo, hi, ptr, stream):
            try:
                torch.cuda.synchronize()                   # a real consumer would queue device work on `stream`
                off = ptr - ring.data_ptr()
                assert off % W == 0 and off // W == w % 3   # slot rotation
                assert ring[off:off + hi - lo].cpu().numpy().tobytes() == x[lo:hi].tobytes(), w
            except Exception as exc:
                errors0.append(exc)
            seen.append((w, lo, hi))
            return 0
        st = ar.decode_stream(0, N, ring, W, consumer=consumer)
        assert not errors0, errors0
        assert [s[0] for s in seen] == list(range(st["n_windows"])) and seen[-1][2] == N and st["bad_blocks"] == 0
        # a sub-range that starts at a window boundary in the middle of the file, two slots
        seen.clear()
        ring2 = ar.new_output(2 * W)
        lo0 = 5 * W

        errors = []

        def consumer2(w, lo, hi, ptr, stream):
            try:                                           # an exception inside a ctypes callback would be swallowed
                torch.cuda.synchronize()
                off = ptr - ring2.data_ptr()
                assert lo == lo0 + w * W and ring2[off:off + hi - lo].cpu().numpy().tobytes() == x[lo:hi].tobytes(), w
            except Exception as exc:
                errors.append(exc)
            seen.append(w)
            return 1 if w == 1 else 0                     # the consumer stops the stream
        with pytest.raises(AceapexError) as e:
            ar.decode_stream(lo0, N, ring2, W, consumer=consumer2)
        assert not errors, errors
        assert e.value.name == "E_ARG" and seen == [0, 1]
        ar.check()
        for bad_args in ((0, N, ring, W + 1), (W // 2, N, ring, W), (0, N, ring[:W // 2], W)):
            with pytest.raises(AceapexError):
                ar.decode_stream(*bad_args)
        # the stream left no resident slot behind: a plain range decode afterwards rebuilds its sources itself
        check_range(ar, x, 5 * W + 3, min(N, 7 * W + 5))
