"""Parity at BASELINE.json's full size: configs[1] (1 GiB synthetic FASTQ, 16 KB blocks), decoded by the calls and in the
launch configuration bench.py times, against the oracle's decode of the same archive (every byte: the oracle finishes
1 GiB in about 15 s) and, for range decode and reads, against the oracle's bytes at sampled windows and reads."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def full():
    import bench
    from oracle import acx_oracle as O
    from paper_2606_18900_b200.aceapex import Archive
    x, a = bench.make_input(1 << 30)                # bench.py's workload: same seed, same encoder settings
    want = np.asarray(O.decode(a))
    assert want.size == (1 << 30) and np.array_equal(want, np.asarray(x))
    ar = Archive(a)
    yield ar, want
    ar.close()


def test_decode_all_every_byte(full):
    ar, want = full
    w = torch.from_numpy(want).cuda()
    for schedule in (None, "flags"):
        out = ar.decode_all(schedule=schedule)
        ar.check()
        assert out.numel() == want.size
        assert torch.equal(out, w), schedule
        assert ar.verify_fnv(out) == 0
        del out


def test_sampled_windows_and_reads(full):
    from paper_2606_18900_b200 import datagen
    ar, want = full
    N = want.size
    rng = np.random.default_rng(11)
    spans = [(0, 1 << 20), (N - (1 << 20) - 12345, N), (N // 2 + 7, N // 2 + 7 + (64 << 20))]
    spans += [(int(lo), int(lo) + int(n)) for lo, n in zip(rng.integers(0, N - (8 << 20), 6), rng.integers(1, 8 << 20, 6))]
    for lo, hi in spans:
        got = ar.decode_range(lo, hi).cpu().numpy()
        ar.check()
        assert np.array_equal(got, want[lo:hi]), (lo, hi)
    idx = datagen.fastq_index(N)
    for n in (1, 3, 700, 5000):
        ids = rng.integers(0, idx.size, n).astype(np.uint64)
        got = ar.decode_reads(idx, ids).cpu().numpy()
        ar.check()
        _, offs = ar.reads_bytes(idx, ids)
        for k, r in enumerate(ids):
            o, ln = int(idx[r]) & ((1 << 40) - 1), int(idx[r]) >> 40
            assert np.array_equal(got[int(offs[k]):int(offs[k]) + ln], want[o:o + ln]), (n, k, int(r))
