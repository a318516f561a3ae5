import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def fastq_4m():
    """configs[0]: 4 MiB synthetic FASTQ, seed 1, 1 Mbp reference."""
    from paper_2606_18900_b200 import datagen
    return datagen.fastq(1, 4 << 20, 1_000_000)


@pytest.fixture(scope="session")
def fastq_4m_archive(fastq_4m):
    from paper_2606_18900_b200 import encoder
    return encoder.encode(fastq_4m, block_size=16384)


@pytest.fixture(scope="session")
def fasta_2m():
    from paper_2606_18900_b200 import datagen
    return datagen.fasta(3, 2 << 20)


@pytest.fixture(scope="session")
def fasta_2m_archive(fasta_2m):
    from paper_2606_18900_b200 import encoder
    return encoder.encode(fasta_2m, block_size=16384)
