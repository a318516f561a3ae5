"""The multithreaded CPU baseline (oracle/acx_mt.c) against the original bytes and the oracle."""
import numpy as np
import pytest

from acx_build import build
from oracle import acx_mt, acx_oracle as O


@pytest.mark.parametrize("threads", [1, 3, 8])
def test_fastq_and_fasta(fastq_4m, fastq_4m_archive, fasta_2m, fasta_2m_archive, threads):
    assert np.array_equal(acx_mt.decode(fastq_4m_archive, threads=threads), fastq_4m)
    assert np.array_equal(acx_mt.decode(fasta_2m_archive, threads=threads), fasta_2m)


def test_hand_built_levels_and_overlap():
    blocks = [[(b"a", (0, 7))], [(b"", (0, 8))], [(b"", (8, 8))], [(b"", (16, 3))]]
    a = build(blocks, 27, 3, min_match=3, levels=[0, 1, 2, 3])
    assert acx_mt.decode(a, threads=4).tobytes() == O.decode(a).tobytes() == b"a" * 27
    lit = bytes((i * 7 + 3) % 251 for i in range(300))
    blocks = [[(lit, (0, 300)), (b"", (10, 4 + 255)), (lit[:255], (1, 4 + 254)), (b"q", None)]]
    N = 300 + 300 + 259 + 255 + 258 + 1
    for raw in [(), (0, 1), (0, 1, 2, 3)]:
        a = build(blocks, N, 11, raw_planes=raw)
        assert acx_mt.decode(a, threads=2).tobytes() == O.decode(a).tobytes()


def test_block_sizes(fastq_4m):
    from paper_2606_18900_b200 import encoder
    x = fastq_4m[:(1 << 20) + 777]
    for bs in (4096, 262144):
        assert np.array_equal(acx_mt.decode(encoder.encode(x, block_size=bs), threads=4), x)
