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
    assert h["log2_seg"] == 14 and h["q_min"] == 64 and h["max_level"] <= 2                 # the encoder's defaults


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


@pytest.mark.parametrize("kw", [dict(q_mode=0), dict(q_mode=1), dict(q_min=0), dict(q_min=2), dict(q_min=300, q_mode=1),
                                dict(block_size=1 << 20), dict(block_size=65536, log2_seg=12), dict(block_size=4096, log2_seg=9),
                                dict(block_size=1 << 18, q_mode=0, max_level=2)])
def test_encoder_options_of_version_3(fastq_4m, fasta_2m, kw):
    """Literal classes, pair symbols and segment sizes (FORMAT.md §1.5-1.7) on FASTQ and FASTA, against the original bytes."""
    for x in (fastq_4m[:(1 << 20) + 4321], fasta_2m[:(1 << 20) + 77]):
        a = encoder.encode(x, **kw)
        h = O.header(a)
        assert np.array_equal(O.decode(a), x)
        assert h["log2_seg"] == kw.get("log2_seg", min(h["log2_bs"], 14)) and h["q_min"] == kw.get("q_min", 64)
        if "q_mode" in kw and h["total_litq"]:
            assert h["q_mode"] == kw["q_mode"]
        if h["log2_bs"] > h["log2_seg"]:
            assert h["n_segs"] > h["n_blocks"]


def test_incompressible_and_huge_runs_are_cut_into_segments():
    """A literal run longer than a segment may hold (16384 literal bytes) and a match longer than a segment."""
    rng = np.random.default_rng(5)
    noise = rng.integers(0, 256, 100_000, dtype=np.uint8)
    x = np.concatenate([noise, np.full(200_000, 65, np.uint8), noise[:50_000], np.tile(noise[:3000], 30)])
    for bs in (1 << 20, 1 << 16, 1 << 14):
        a = encoder.encode(x, block_size=bs)
        assert np.array_equal(O.decode(a), x)
    h = O.header(encoder.encode(x, block_size=1 << 20))
    assert h["n_blocks"] == 1 and h["n_segs"] >= 10 and h["q_mode"] == 0          # 65,536 distinct pairs: byte mode


def test_src_window_option(fasta_2m):
    a = encoder.encode(fasta_2m, src_window=65536)
    assert np.array_equal(O.decode(a), fasta_2m)
    n_segs = O.header(a)["n_segs"]
    for sg in range(0, n_segs, 7):
        blk = O.segment(a, sg)
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
    replay of the stage-level streams reproduces the original bytes of the segment."""
    h = O.header(fastq_4m_archive)
    BS = 1 << h["log2_bs"]
    for b in (0, 1, 100, 255):
        s0, s1, level = O.block_segs(fastq_4m_archive, b)
        ends = []
        for sg in range(s0, s1):
            k = O.segment(fastq_4m_archive, sg)
            assert k["block"] == b and k["level"] == level
            assert int(k["lit_len"].sum()) == k["n_lit"] == len(k["lit"]) == k["n_lit_a"] + k["n_lit_q"]
            longq = k["lit_len"] >= h["q_min"]
            assert int(k["lit_len"][longq].sum()) == k["n_lit_q"] and int(k["lit_len"][~longq].sum()) == k["n_lit_a"]
            assert int(k["lit_len"].sum() + k["match_len"].sum()) == k["out_end"] - k["out_start"]
            assert (np.diff(k["out_pos"].astype(np.int64)) >= 0).all()
            assert (k["out_pos"] - k["out_start"] < (1 << h["log2_seg"])).all()          # FORMAT.md §1.5: command starts
            assert np.array_equal(k["out_pos"], k["out_start"] + np.concatenate([[0], np.cumsum(k["lit_len"] + k["match_len"])[:-1]]).astype(np.uint64))
            out = bytearray(fastq_4m[:k["out_start"]].tobytes()) + bytearray(k["out_end"] - k["out_start"])   # earlier bytes given
            dst, lp = k["out_start"], 0
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
            assert dst == k["out_end"] and bytes(out[k["out_start"]:dst]) == fastq_4m[k["out_start"]:dst].tobytes()
            ends.append((k["out_start"], k["out_end"]))
        assert ends[0][0] == b * BS and ends[-1][1] == min(BS * (b + 1), h["N"])
        assert all(a[1] == c[0] for a, c in zip(ends, ends[1:]))


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
