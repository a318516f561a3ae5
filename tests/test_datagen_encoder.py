"""Host-side checks of the input generators and of the encoder's determinism."""
import numpy as np

from oracle import acx_oracle as O
from paper_2606_18900_b200 import datagen, encoder


def test_fastq_shape(fastq_4m):
    lines = fastq_4m.tobytes().split(b"\n")
    assert lines[0] == b"@SIM.1 1/1" and lines[2] == b"+" and lines[4] == b"@SIM.2 2/1"
    for r in range(0, 2000, 97):
        hdr, bases, plus, quals = lines[4 * r:4 * r + 4]
        assert hdr == b"@SIM.%d %d/1" % (r + 1, r + 1)
        assert len(bases) == 150 and set(bases) <= set(b"ACGTN")
        assert plus == b"+" and len(quals) == 150
        assert min(quals) >= 33 + 2 and max(quals) <= 33 + 41
    q = np.array([list(lines[4 * r + 3]) for r in range(3000)], dtype=np.float64) - 33
    assert abs(q[:, 0].mean() - 36) < 0.5 and abs(q[:, 149].mean() - 28) < 0.5     # mean drops from 36 to 28
    assert 3.3 < q[:, 75].std() < 4.5                                               # sd 4 (clipped, rounded)
    n_frac = (fastq_4m == ord("N")).sum() / (fastq_4m.size * 150 / 323)
    assert 0.0005 < n_frac < 0.002


def test_fastq_windows_and_seed(fastq_4m):
    for lo, hi in [(0, 1), (12345, 99999), (4194000, 4194304), (322, 324)]:
        assert np.array_equal(datagen.fastq(1, 4 << 20, 1_000_000, lo=lo, hi=hi), fastq_4m[lo:hi])
    assert not np.array_equal(datagen.fastq(2, 1 << 16, 1_000_000), fastq_4m[:1 << 16])
    assert np.array_equal(datagen.fastq(1, 4 << 20, 1_000_000, threads=1), fastq_4m)


def test_fastq_index(fastq_4m):
    idx = datagen.fastq_index(4 << 20)
    assert idx.size == datagen.fastq_n_reads(4 << 20)
    off = (idx & ((1 << 40) - 1)).astype(np.int64)
    ln = (idx >> 40).astype(np.int64)
    for r in (0, 1, 9, 10, 999, 1000, idx.size - 1):
        rec = fastq_4m[off[r]:off[r] + ln[r]].tobytes()
        assert rec.startswith(b"@SIM.%d %d/1\n" % (r + 1, r + 1)) and rec.endswith(b"\n") and rec.count(b"\n") == 4
    assert off[-1] + ln[-1] <= 4 << 20


def test_fasta_shape(fasta_2m):
    text = fasta_2m.tobytes()
    assert len(text) == 2 << 20
    lines = text.split(b"\n")
    heads = [l for l in lines if l.startswith(b">")]
    assert heads == [b">chr%d" % i for i in range(1, 25)]
    body = [l for l in lines if not l.startswith(b">")]
    assert max(len(l) for l in body) == 60
    assert set(b"".join(body)) <= set(b"ACGTN")
    assert np.array_equal(datagen.fasta(3, 2 << 20), fasta_2m)


def test_region_index():
    idx = datagen.region_index(3, 1 << 20, 1000, 150)
    off = idx & np.uint64((1 << 40) - 1)
    assert ((idx >> np.uint64(40)) == 150).all() and int(off.max()) <= (1 << 20) - 150
    assert np.array_equal(idx, datagen.region_index(3, 1 << 20, 1000, 150))


def test_encoder_is_deterministic_across_thread_counts(fastq_4m):
    x = fastq_4m[:3 << 20]
    a1 = encoder.encode(x, threads=1, chunk_log2=18, batch_chunks=4)
    a4 = encoder.encode(x, threads=4, chunk_log2=18, batch_chunks=4)
    assert np.array_equal(a1, a4)
    assert np.array_equal(O.decode(a4), x)
