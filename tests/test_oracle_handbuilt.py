"""Pins of the oracle's LZ copy semantics, block partition and level invariant on hand-built archives.

Archives are assembled by tests/acx_build.py (FORMAT.md restated in Python, own rANS encoder); the expected outputs
are written by hand below.  FORMAT.md §2 reduces to textbook LZ77 semantics (copy `len` bytes from an earlier
position, ascending, byte by byte), so every expected string can be checked by eye."""
import pytest

from acx_build import build, lz_reference
from oracle import acx_oracle as O


def dec(blocks, N, log2_bs, **kw):
    return bytes(O.decode(build(blocks, N, log2_bs, **kw)))


def test_literals_only_single_block():
    assert dec([[(b"hello", None)]], 5, 3) == b"hello"


def test_rle_one_byte_period_across_blocks():
    # 'a', an in-block run (src = dst-1), then every block copies its predecessor.  Blocks of 8 bytes, N = 27 (ragged tail).
    blocks = [[(b"a", (0, 7))], [(b"", (0, 8))], [(b"", (8, 8))], [(b"", (16, 3))]]
    # each block reads a match byte of its predecessor -> levels must increase (FORMAT.md §3)
    assert dec(blocks, 27, 3, min_match=3, levels=[0, 1, 2, 3]) == b"a" * 27
    with pytest.raises(O.OracleError):
        dec(blocks, 27, 3, min_match=3, levels=[0, 1, 1, 2])


def test_self_overlap_needs_its_seed_in_the_own_block():
    # FORMAT.md §3 (c): a self-overlapping match (src + len > dst) starts in its own block.  src = 7, dst = 8, len = 8
    # would continue the run of block 0 from outside block 1: rejected.
    with pytest.raises(O.OracleError) as e:
        dec([[(b"a", (0, 7))], [(b"", (7, 8))]], 16, 3, min_match=3, levels=[0, 1])
    assert e.value.name == "E_CORRUPT"
    # the same bytes with the run restarted by a literal inside block 1 are fine
    assert dec([[(b"a", (0, 7))], [(b"a", (8, 7))]], 16, 3, min_match=3, levels=[0, 0]) == b"a" * 16


def test_period_three_overlap():
    # "abc" + copy 10 from position 0: abc abc abc abc a
    assert dec([[(b"abc", (0, 10))]], 13, 4) == b"abcabcabcabca"


def test_source_ends_exactly_at_dst():
    # src + len == dst: the boundary between the non-overlapping and the self-overlapping case
    assert dec([[(b"wxyz", (0, 4))]], 8, 3) == b"wxyzwxyz"


def test_match_ends_at_block_end_and_match_starts_block():
    # block 0 (8 B): "abcd" + copy(0,4) ends exactly at the block end; block 1 starts with a match, then a literal tail
    blocks = [[(b"abcd", (0, 4))], [(b"", (2, 5)), (b"XYZ", None)]]
    # block 1 reads bytes 4..6, match bytes of block 0 -> level 1
    assert dec(blocks, 16, 3, levels=[0, 1]) == b"abcdabcd" + b"cdabc" + b"XYZ"


def test_source_spans_two_blocks():
    # bytes 6..10 straddle blocks 0|1
    blocks = [[(b"01234567", None)], [(b"89ab", (6, 4))], [(b"", (6, 5)), (b"!!!", None)]]
    assert dec(blocks, 24, 3) == b"0123456789ab6789" + b"6789a" + b"!!!"


def test_block_with_zero_literals_and_block_with_zero_matches():
    blocks = [[(b"ACGTACGT", None)], [(b"", (0, 4)), (b"", (4, 4))]]
    assert dec(blocks, 16, 3) == b"ACGTACGTACGTACGT"


def test_far_source_levels():
    # block 2 copies match bytes of block 1 -> needs level(2) > level(1)
    blocks = [[(b"ABCDEFGH", None)], [(b"", (0, 8))], [(b"", (8, 8))]]
    assert dec(blocks, 24, 3, levels=[0, 0, 1]) == b"ABCDEFGH" * 3
    with pytest.raises(O.OracleError) as e:
        dec(blocks, 24, 3, levels=[0, 0, 0])
    assert e.value.name == "E_LEVEL"


def test_literal_bytes_of_a_higher_level_block_violate_levels():
    # FORMAT.md §3 (a): literal bytes may only be read from blocks whose level is NOT HIGHER than the reader's.  Block 1
    # copies the eight literal bytes of block 0.  With level(0) = 1 and level(1) = 0 the reader sits below its source: the
    # (level, index) dispatch order of the flag schedules would start block 1 before block 0 -> rejected.
    blocks = [[(b"ABCDEFGH", None)], [(b"", (0, 8))]]
    with pytest.raises(O.OracleError) as e:
        dec(blocks, 16, 3, levels=[1, 0])
    assert e.value.name == "E_LEVEL"
    # the same bytes with legal levels (equal, or the reader higher) decode to the hand-written output
    for lv in ([0, 0], [1, 1], [0, 1], [2, 3]):
        assert dec(blocks, 16, 3, levels=lv) == b"ABCDEFGH" * 2
    # a source two blocks back at a higher level is rejected as well; one literal byte is enough
    blocks3 = [[(b"ABCDEFGH", None)], [(b"IJKLMNOP", None)], [(b"xyz", (7, 5))]]
    assert dec(blocks3, 24, 3, levels=[0, 0, 0]) == b"ABCDEFGHIJKLMNOP" + b"xyz" + b"HIJKL"
    with pytest.raises(O.OracleError) as e:
        dec(blocks3, 24, 3, levels=[1, 0, 0])       # byte 7 is a literal byte of block 0 (level 1 > 0)
    assert e.value.name == "E_LEVEL"
    with pytest.raises(O.OracleError) as e:
        dec(blocks3, 24, 3, levels=[0, 2, 1])       # bytes 8..11 are literal bytes of block 1 (level 2 > 1)
    assert e.value.name == "E_LEVEL"


def test_in_block_match_bytes_as_source_violate_levels():
    # second match reads bytes produced by the first match of the same block: forbidden by FORMAT.md §3
    blocks = [[(b"abcd", (0, 4)), (b"", (4, 4)), (b"zzzz", None)]]
    with pytest.raises(O.OracleError) as e:
        dec(blocks, 16, 4)
    assert e.value.name == "E_LEVEL"
    # the same bytes are fine when the level check is off (pure FORMAT.md §2 semantics)
    assert bytes(O.decode(build(blocks, 16, 4), check_levels=False)) == b"abcdabcdabcdzzzz"


def test_self_overlap_seed_must_be_literal_but_own_output_is_exempt():
    # literal "xy", copy(0, 9): seed = [0,2) literal; bytes >= dst are produced by the match itself (exempt)
    assert dec([[(b"xy", (0, 9)), (b"END", None)]], 14, 4) == b"xyxyxyxyxyx" + b"END"


@pytest.mark.parametrize("N", [0, 1, 7, 8, 9])
def test_sizes_around_a_block(N):
    data = b"abcdefghi"[:N]
    blocks = [[(data[i:i + 8], None)] for i in range(0, N, 8)]
    assert dec(blocks, N, 3) == data


def test_long_literal_and_long_match_escapes():
    # lit_len >= 255 and match_len - min_match >= 255 use EXT (FORMAT.md §1.4), CMD escapes before MLEN escapes
    lit = bytes((i * 7 + 3) % 251 for i in range(300))
    blocks = [[(lit, (0, 300)), (b"", (10, 4 + 255)), (lit[:255], (1, 4 + 254)), (b"q", None)]]
    N = 300 + 300 + 259 + 255 + 258 + 1
    exp = lit + lit + lit[10:10 + 259] + lit[:255] + lit[1:1 + 258] + b"q"
    assert dec(blocks, N, 11) == exp


def test_offsets_use_all_planes_coded_or_raw():
    lit = bytes(range(256)) * 2
    blocks = [[(lit, (0x101, 8)), (b"", (0x1, 8)), (b"", (0x1F0, 16))]]
    exp = lit + lit[0x101:0x109] + lit[1:9] + lit[0x1F0:0x200]
    for raw in [(), (0,), (0, 1), (0, 1, 2, 3)]:
        assert dec(blocks, len(exp), 10, raw_planes=raw) == exp


def test_python_reference_agrees_on_a_mixed_case():
    blocks = [[(b"GATTACA!", None)], [(b"", (1, 3 + 1)), (b"NN", (12, 2))], [(b"", (3, 8))]]
    exp = lz_reference(blocks, 24, 3)
    assert exp == b"GATTACA!" + b"ATTA" + b"NN" + b"NN" + b"TACA!ATT"
    assert dec(blocks, 24, 3, min_match=2, levels=[0, 0, 1]) == exp


def test_fnv_section_checked():
    blocks = [[(b"ABCDEFGH", None)], [(b"", (0, 8))]]
    exp = b"ABCDEFGH" * 2
    assert dec(blocks, 16, 3, with_fnv=True, expected=exp) == exp
    with pytest.raises(O.OracleError):
        dec(blocks, 16, 3, with_fnv=True, expected=b"ABCDEFGHABCDEFGX")
    # FNV-1a 64 published test vectors (Fowler/Noll/Vo): "" and "a"
    assert O.fnv1a64(b"") == 0xCBF29CE484222325
    assert O.fnv1a64(b"a") == 0xAF63DC4C8601EC8C
    assert O.fnv1a64(b"foobar") == 0x85944171F73967E8


def _mut(off, val):
    def f(buf):
        buf[off] = val
    return f


def test_corrupt_archives_are_rejected():
    blocks = [[(b"abcd", (0, 4))], [(b"", (2, 5)), (b"XYZ", None)]]
    good = build(blocks, 16, 3, levels=[0, 1])
    assert bytes(O.decode(good)) == b"abcdabcdcdabcXYZ"
    with pytest.raises(O.OracleError) as e:
        O.decode(build(blocks, 16, 3, levels=[0, 1], mutate=_mut(0, 0x42)))
    assert e.value.name == "E_MAGIC"
    with pytest.raises(O.OracleError) as e:
        O.decode(build(blocks, 16, 3, levels=[0, 1], mutate=_mut(8, 1)))   # version 1 archives are not readable
    assert e.value.name == "E_VERSION"
    with pytest.raises(O.OracleError) as e:
        O.decode(good[:-16])
    assert e.value.name == "E_TRUNCATED"
    with pytest.raises(O.OracleError):
        O.decode(good[:100])
    # forward reference: src >= dst
    with pytest.raises(O.OracleError) as e:
        dec([[(b"abcd", (4, 4))]], 8, 3)
    assert e.value.name == "E_CORRUPT"
    # match crossing the block end
    with pytest.raises(O.OracleError):
        dec([[(b"abcd", (0, 5))], [(b"xyz", None)]], 12, 3)
    # a flipped payload byte must trip the rANS integrity checks (final states / word count) or a format check
    h = O.header(good)
    bad = bytearray(good)
    bad[h["payload_off"] + 1] ^= 0x5A  # inside the initial state of lane 0
    with pytest.raises(O.OracleError):
        O.decode(bytes(bad))


def test_word_offsets_of_the_rans_head_are_checked():
    # FORMAT.md §1.5: word_off[0] = 0, non-decreasing, word_off[32] = n_words; every state consumes exactly its stream
    lit0, lit1 = bytes((i * 37 + 11) % 251 for i in range(252)), bytes((i * 91 + 5) % 241 for i in range(232))
    blocks = [[(lit0, (0, 4))], [(b"", (2, 24)), (lit1, None)]]
    N = 512
    good = build(blocks, N, 8, levels=[0, 0])
    exp = O.decode(good).tobytes()
    assert exp == lit0 + lit0[:4] + lit0[2:26] + lit1
    h = O.header(good)
    po = h["payload_off"]
    offs = [int.from_bytes(good[po + 8 * k + 4:po + 8 * k + 8], "little") for k in range(32)]
    assert offs[0] == 0 and offs == sorted(offs) and offs[-1] > 0      # the block does use words
    for k, delta in ((0, 1), (5, 1), (31, -1)):
        bad = bytearray(good)
        v = offs[k] + delta
        if v < 0:
            continue
        bad[po + 8 * k + 4:po + 8 * k + 8] = v.to_bytes(4, "little")
        with pytest.raises(O.OracleError):
            O.decode(bytes(bad))
