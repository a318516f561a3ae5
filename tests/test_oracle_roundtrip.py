"""decode(encode(x)) == x against the ORIGINAL bytes: the absolute pin of the whole decoder ("bit-perfect
... XXH3-64 for CPU paths ... against the original bytes").  It does not depend on the oracle being right."""
import itertools

import numpy as np
import pytest
import xxhash
from hypothesis import given, settings
from hypothesis import strategies as st

from oracle import acx_oracle as O
from paper_2606_18900_b200 import encoder


def rt(data, **kw):
    data = np.frombuffer(bytes(data), dtype=np.uint8)
    a = encoder.encode(data, **kw)
    out = O.decode(a)           # check_levels=True: FORMAT.md §3 invariant and FNV verified as well
    assert out.tobytes() == data.tobytes()
    return a


def test_config0_fastq_bit_exact_and_xxh3(fastq_4m, fastq_4m_archive):
    out = O.decode(fastq_4m_archive)
    assert np.array_equal(out, fastq_4m)
    assert xxhash.xxh3_64_intdigest(out.tobytes()) == xxhash.xxh3_64_intdigest(fastq_4m.tobytes())
    h = O.header(fastq_4m_archive)
    assert h["N"] == 4 << 20 and h["n_blocks"] == 256 and h["log2_bs"] == 14 and h["min_match"] == 4


def test_fasta_bit_exact(fasta_2m, fasta_2m_archive):
    assert np.array_equal(O.decode(fasta_2m_archive), fasta_2m)


def test_brute_force_all_binary_strings():
    # every string over {a,b} up to length 11, block sizes 8 and 16 (matches, overlaps, block splits all occur)
    for n in range(0, 12):
        for bits in itertools.product(b"ab", repeat=n):
            for bs in (8, 16):
                rt(bytes(bits), block_size=bs)


@pytest.mark.parametrize("bs", [8, 64, 4096, 16384, 65536])
def test_sizes_around_block_boundaries(bs):
    rng = np.random.default_rng(bs)
    base = rng.integers(65, 69, 3 * bs + 5, dtype=np.uint8)
    base[bs // 2:bs] = base[:bs - bs // 2]      # some repetition
    for n in (1, bs - 1, bs, bs + 1, 2 * bs, 3 * bs + 5):
        rt(base[:n], block_size=bs)


def test_long_runs_and_periods_cross_many_blocks():
    rt(b"N" * 100000, block_size=4096)
    rt((b"ACGTTGCA" * 7 + b"\n") * 3000, block_size=16384)
    rt(b"x" + b"\0" * 70000 + b"y", block_size=1024)


@pytest.mark.parametrize("max_level", [0, 1, 3, 7])
def test_level_cap_is_respected(fastq_4m, max_level):
    a = encoder.encode(fastq_4m[:1 << 20], max_level=max_level)
    assert O.header(a)["max_level"] <= max_level
    assert np.array_equal(O.decode(a), fastq_4m[:1 << 20])


def test_src_window_option(fasta_2m):
    a = encoder.encode(fasta_2m, src_window=65536)
    assert np.array_equal(O.decode(a), fasta_2m)
    n_blocks = O.header(a)["n_blocks"]
    for b in range(0, n_blocks, 7):
        blk = O.block(a, b)
        dst = blk["out_pos"][:blk["n_match"]] + blk["lit_len"][:blk["n_match"]]
        assert ((dst - blk["src"]) <= 65536).all()


@settings(max_examples=150, deadline=None)
@given(st.lists(st.tuples(st.binary(min_size=1, max_size=12), st.integers(1, 40)), min_size=0, max_size=12),
       st.sampled_from([8, 32, 256]))
def test_hypothesis_repetitive(parts, bs):
    data = b"".join(p * k for p, k in parts)
    rt(data, block_size=bs)


def test_stage_view_is_consistent_with_decode(fastq_4m, fastq_4m_archive):
    """Invariants of the scan: sums, counts, monotone positions; and an independent Python byte-serial
    replay of the stage-level streams reproduces the original block."""
    h = O.header(fastq_4m_archive)
    BS = 1 << h["log2_bs"]
    for b in (0, 1, 100, 255):
        k = O.block(fastq_4m_archive, b)
        assert int(k["lit_len"].sum()) == k["n_lit"] == len(k["lit"])
        assert int(k["lit_len"].sum() + k["match_len"].sum()) == min(BS, h["N"] - b * BS)
        assert (np.diff(k["out_pos"].astype(np.int64)) >= 0).all()
        assert np.array_equal(k["lit_pos"], np.concatenate([[0], np.cumsum(k["lit_len"])[:-1]]).astype(np.uint32))
        assert np.array_equal(k["out_pos"], b * BS + np.concatenate([[0], np.cumsum(k["lit_len"] + k["match_len"])[:-1]]).astype(np.uint64))
        out = bytearray(fastq_4m[:b * BS].tobytes()) + bytearray(BS)    # earlier blocks given, this block replayed
        dst, lp = b * BS, 0
        for c in range(k["n_cmd"]):
            ll, ml = int(k["lit_len"][c]), int(k["match_len"][c])
            out[dst:dst + ll] = k["lit"][lp:lp + ll].tobytes()
            dst += ll
            lp += ll
            if c < k["n_match"]:
                s = int(k["src"][c])
                assert s < dst
                for i in range(ml):
                    out[dst + i] = out[s + i]
                dst += ml
        assert bytes(out[b * BS:dst]) == fastq_4m[b * BS:dst].tobytes()


def test_periodic_data_small_blocks_keep_overlaps_in_their_block():
    """FORMAT.md §3 (c) under stress: mutated periodic data, periods around the block size.  The oracle rejects any
    self-overlapping match whose source starts outside its block, so a clean decode is the check.  (Seeds 8, 12, 29, 39,
    53 of this recipe caught an encoder that extended a match cut to exactly one period backwards into an overlap.)"""
    from paper_2606_18900_b200 import encoder
    for seed in range(120):
        rng = np.random.default_rng(seed)
        period, alpha, n = int(rng.integers(3, 40)), int(rng.integers(2, 5)), int(rng.integers(1500, 5000))
        pat = rng.integers(65, 65 + alpha, period, dtype=np.uint8)
        x = np.tile(pat, n // period + 1)[:n].copy()
        m = rng.random(n) < rng.uniform(0.002, 0.03)
        x[m] = rng.integers(65, 65 + alpha + 1, int(m.sum()), dtype=np.uint8)
        bs = int(rng.choice([32, 64, 128, 256, 1024]))
        a = encoder.encode(x, block_size=bs, chunk_log2=11, batch_chunks=2)
        assert np.array_equal(O.decode(a), x), (seed, bs)
