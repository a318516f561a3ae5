"""BASELINE.json configs at (or near) full size on the GPU, driver-runnable: positions above 2^32 with 5-byte offsets
(section 5: "a 4 GB uint32 overflow ... size and offset fields migrated to 64-bit"), configs[2] (3.1 GB FASTA +
10^6 region reads), the block-size sweep of configs[4] on the 1 GiB FASTQ, and a file larger than its ring through
aceapex_decode_stream (configs[3] in small: the 50 GiB run itself is `python -m paper_2606_18900_b200.report --config 3`).

What each case is compared with: the ORIGINAL bytes (regenerated from the seed), every byte, on the device; the archive's
per-block FNV-1a table; and the oracle's decode where stated (the 5 GiB case: every byte)."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

G = 1 << 30


def equal_on_device(out, x, chunk=1 << 30):
    """out: CUDA uint8 tensor; x: numpy uint8 array of the same length; compared chunk by chunk on the device."""
    assert out.numel() == x.size
    for lo in range(0, x.size, chunk):
        hi = min(x.size, lo + chunk)
        if not torch.equal(out[lo:hi], torch.from_numpy(x[lo:hi]).to(out.device)):
            return False
    return True


@pytest.fixture(scope="module")
def fasta_5g():
    from paper_2606_18900_b200 import datagen, encoder
    from paper_2606_18900_b200.aceapex import Archive
    x = datagen.fasta(4, 5 * G)                      # the configs[3] generator (seed 4), 5 GiB: positions need 33 bits
    a = encoder.encode(x, block_size=16384)
    ar = Archive(a)
    yield ar, x, a
    ar.close()


def test_positions_above_4GiB_every_byte_vs_oracle_and_original(fasta_5g):
    from oracle import acx_oracle as O
    ar, x, a = fasta_5g
    info = ar.info()
    assert info["raw_bytes"] == 5 * G and info["offset_width"] == 5 and info["n_blocks"] == 5 * G // 16384
    out = ar.decode_all()
    ar.check()
    assert ar.verify_fnv(out) == 0
    assert equal_on_device(out, x)                                   # the original bytes
    want = O.decode(a, check_levels=False)                          # the oracle, every byte (about 20 s on one core)
    assert np.array_equal(want, x)
    assert equal_on_device(out, want)
    for sched in ("flags", "fused"):
        out.zero_()
        ar.decode_all(out, schedule=sched)
        ar.check()
        assert ar.verify_fnv(out) == 0 and equal_on_device(out[4 * G:], x[4 * G:])


def test_ranges_and_reads_above_4GiB(fasta_5g):
    ar, x, a = fasta_5g
    N = x.size
    # windows whose lo is above 2^32: block aligned, 16-byte aligned, odd; a window that straddles 2^32; the file's end
    for lo, n in ((4 * G + 16384 * 1000, 32 << 20), (4 * G + 16 * 12345, 8 << 20), (4 * G + 7777777, (4 << 20) + 3), (4 * G - (3 << 20) - 5, 6 << 20),
                  (N - (5 << 20) - 1, (5 << 20) + 1), (4 * G + 123, 1), (4 * G + (700 << 20), 200)):
        got = ar.decode_range(lo, lo + n)
        ar.check()
        assert got.cpu().numpy().tobytes() == x[lo:lo + n].tobytes(), (lo, n)
    rng = np.random.default_rng(4)
    off = rng.integers(4 * G, N - 150, 5000).astype(np.uint64)       # 150-byte region reads, every offset above 2^32
    idx = off | (np.uint64(150) << np.uint64(40))
    for n in (1, 37, 4096):
        ids = rng.integers(0, idx.size, n).astype(np.uint64)
        got = ar.decode_reads(idx, ids).cpu().numpy()
        ar.check()
        for k in range(0, n, 11):
            o = int(off[ids[k]])
            assert got[150 * k:150 * k + 150].tobytes() == x[o:o + 150].tobytes(), (n, k)


def test_file_larger_than_its_ring(fasta_5g):
    """configs[3] in small: 5 GiB through a ring of four 256 MiB slots; the library's device FNV consumer checks every block."""
    ar, x, a = fasta_5g
    W = 256 << 20
    ring = ar.new_output(4 * W)
    st = ar.decode_stream(0, x.size, ring, W)
    assert st["n_windows"] == 20 and st["n_slots"] == 4 and st["bytes"] == x.size and st["bad_blocks"] == 0
    assert st["peak_device_bytes"] < ar.info()["archive_bytes"] + 4 * W + ar.info()["workspace_bytes"] + 1
    # the last window is still in its slot: compare it with the original bytes
    lo = 19 * W
    assert torch.equal(ring[3 * W:4 * W], torch.from_numpy(x[lo:lo + W]).cuda())
    del ring


def test_config2_genome_and_region_reads():
    """configs[2]: 3.1 GB FASTA (seed 3), whole file against the original bytes and the FNV table; 10^6 region reads of 150
    bytes, batches of 4096 and single reads, sampled against slices of the original."""
    from paper_2606_18900_b200 import datagen, encoder
    from paper_2606_18900_b200.aceapex import Archive
    N = 3_100_000_000
    x = datagen.fasta(3, N)
    ar = Archive(encoder.encode(x, block_size=16384))
    assert ar.info()["n_blocks"] == 189_209 and ar.info()["offset_width"] == 4
    out = ar.decode_all()
    ar.check()
    assert ar.verify_fnv(out) == 0 and equal_on_device(out, x)
    del out
    idx = datagen.region_index(3, N, 1_000_000, 150)
    off = (idx & np.uint64((1 << 40) - 1)).astype(np.int64)
    rng = np.random.default_rng(2)
    for n in (4096, 4096, 1, 1, 1):
        ids = rng.integers(0, idx.size, n).astype(np.uint64)
        got = ar.decode_reads(idx, ids).cpu().numpy()
        ar.check()
        for k in range(0, n, 13):
            o = int(off[ids[k]])
            assert got[150 * k:150 * k + 150].tobytes() == x[o:o + 150].tobytes(), (n, k)
    ar.close()


@pytest.mark.parametrize("bs", [4096, 8192, 16384, 65536, 262144, 1 << 20])
def test_config4_block_size_sweep_on_the_1GiB_fastq(bs):
    """configs[4]: the configs[1] FASTQ at every block size of the sweep, all three schedules, against the original bytes."""
    import bench
    from paper_2606_18900_b200 import datagen, encoder
    from paper_2606_18900_b200.aceapex import Archive
    x = datagen.fastq(2, 1 << 30, 50_000_000)
    ar = Archive(encoder.encode(x, block_size=bs))
    info = ar.info()
    assert info["n_blocks"] == (1 << 30) // bs and info["n_segments"] >= (1 << 30) // max(bs, 16384)
    xt = torch.from_numpy(x).cuda()
    for sched in (None, "flags", "fused"):
        out = ar.decode_all(schedule=sched)
        ar.check()
        assert torch.equal(out, xt), (bs, sched)
        assert ar.verify_fnv(out) == 0
        del out
    lo = (1 << 29) + 12345
    assert torch.equal(ar.decode_range(lo, lo + (3 << 20)), xt[lo:lo + (3 << 20)])
    ar.check()
    ar.close()
