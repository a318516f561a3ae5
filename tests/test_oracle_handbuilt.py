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
    # FORMAT.md §3 (c): the seed of a self-overlapping match (src + len > dst) is the tail of its own command's literal
    # run.  src = 7, dst = 8, len = 8 would continue the run of block 0 from outside block 1: rejected.
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


# ---------------------------------------------------------------------------------------------- version 3 --------
# Segments (FORMAT.md §1.5), the two literal classes (§1.6) and pair symbols (§1.7).  Expected bytes written by hand.

SEGS3 = [[(b"ABCDEFGHIJ", None)], [(b"KL", (0, 3)), (b"mn", (2, 4))], [(b"", (8, 4)), (b"wxyz123", None)]]
EXP3 = b"ABCDEFGHIJ" + b"KL" + b"ABC" + b"mn" + b"CDEF" + b"IJKL" + b"wxyz123"


def test_block_of_three_segments_and_a_literal_run_cut_at_a_segment_boundary():
    # one block of 32 bytes, SEG = 8.  Segment 0: the run "ABCDEFGHIJ" without a match (a segment may end with a match-less
    # command); segment 1 (out_start 10): "KL" + copy(0, 3) + "mn" + copy(2, 4); segment 2 (out_start 21): copy(8, 4) + "wxyz123".
    assert len(EXP3) == 32
    a = build([SEGS3], 32, 5, log2_seg=3, min_match=2)
    assert bytes(O.decode(a)) == EXP3 == lz_reference([SEGS3], 32, 5)
    h = O.header(a)
    assert (h["n_blocks"], h["n_segs"], h["log2_seg"]) == (1, 3, 3)
    assert O.block_segs(a, 0) == (0, 3, 0)
    s1 = O.segment(a, 1)
    assert (s1["out_start"], s1["out_end"], s1["n_cmd"], s1["n_match"]) == (10, 21, 2, 2)
    assert s1["out_pos"].tolist() == [10, 15] and s1["lit"].tobytes() == b"KLmn" and s1["src"].tolist() == [0, 2]
    assert O.segment(a, 2)["out_end"] == 32 and O.segment(a, 0)["n_match"] == 0


def test_a_command_may_not_start_beyond_SEG_bytes_of_its_segment():
    # SEG = 8: the second command of this single segment would start at segment offset 8
    cmds = [(b"abcd", (0, 4)), (b"", (0, 4)), (b"", (0, 4))]
    assert dec([cmds], 16, 4, log2_seg=4) == b"abcdabcdabcdabcd"
    with pytest.raises(O.OracleError) as e:
        dec([cmds], 16, 4, log2_seg=3)
    assert e.value.name == "E_CORRUPT"
    assert dec([[cmds[:1], cmds[1:]]], 16, 4, log2_seg=3) == b"abcdabcdabcdabcd"      # cut into two segments: legal


def _patch(off, data):
    def f(buf):
        buf[off:off + len(data)] = data
    return f


def test_segment_directory_and_block_table_are_checked():
    blocks = [SEGS3, [(b"", (0, 8))]]
    good = build(blocks, 40, 5, log2_seg=3, min_match=2)
    assert bytes(O.decode(good)) == EXP3 + b"ABCDEFGH"
    h = O.header(good)
    d, bt = h["dir_off"], h["blocktab_off"]
    bad = [
        _patch(d + 32 * 1 + 8, (11).to_bytes(8, "little")),       # out_start of segment 1 moved: segment 0 no longer ends where its commands end
        _patch(d + 32 * 2 + 8, (10).to_bytes(8, "little")),       # out_start not strictly increasing inside the block (segment 1 starts at 10)
        _patch(d + 32 * 3 + 8, (33).to_bytes(8, "little")),       # first segment of block 1 must start at 32
        _patch(d + 32 * 1 + 30, (1).to_bytes(2, "little")),       # level copy differs from the block table
        _patch(d + 32 * 0 + 16, (0).to_bytes(2, "little")),       # n_cmd = 0
        _patch(bt + 8, (4).to_bytes(4, "little")),                # block 1 would own no segment
        _patch(bt + 8, (2).to_bytes(4, "little")),                # segment 2 moved to block 1: its out_start is not a block start
        _patch(bt + 16, (5).to_bytes(4, "little")),               # final entry != n_segs
        _patch(len(good) - 1, b"\x01"),                            # tail pad must be zero
        _patch(72, (2).to_bytes(4, "little")),                    # log2_seg below 3
        _patch(72, (6).to_bytes(4, "little")),                    # log2_seg above log2_bs
    ]
    for m in bad:
        with pytest.raises(O.OracleError):
            O.decode(build(blocks, 40, 5, log2_seg=3, min_match=2, mutate=m))
    with pytest.raises(O.OracleError) as e:
        O.decode(good[:-16])
    assert e.value.name == "E_TRUNCATED"


def test_two_literal_classes_byte_mode():
    # q_min = 4: runs of 4 bytes or more are LITQ, shorter ones LITA (FORMAT.md §1.6).  The two streams are stored apart
    # (LITA = "abXY!", LITQ = "QQQQQ" "RSTUVW"), the output interleaves them in command order.
    cmds = [(b"ab", (0, 2)), (b"QQQQQ", (4, 3)), (b"XY", (4, 4)), (b"RSTUVW", (12, 2)), (b"!", None)]
    exp = b"ab" + b"ab" + b"QQQQQ" + b"QQQ" + b"XY" + b"QQQQ" + b"RSTUVW" + b"XY" + b"!"
    a = build([cmds], len(exp), 5, min_match=2, q_min=4)
    assert bytes(O.decode(a)) == exp == lz_reference([cmds], len(exp), 5)
    s = O.segment(a, 0)
    assert (s["n_lit_a"], s["n_lit_q"], s["n_sym_q"]) == (5, 11, 11)
    assert s["lit_pos"].tolist() == [0, 0, 2, 5, 4]              # position of each run in ITS stream
    assert O.header(a)["total_litq"] == 11
    # with q_min = 0 the same commands put everything into LITA
    a0 = build([cmds], len(exp), 5, min_match=2, q_min=0)
    assert bytes(O.decode(a0)) == exp and O.segment(a0, 0)["n_lit_a"] == 16
    # the class is decided by the header's q_min alone: q_min = 5 classifies these runs (2, 5, 2, 6, 1 bytes) as 4 did and
    # decodes; with q_min = 6 the decoder looks for "QQQQQ" in LITA and the streams no longer add up
    assert bytes(O.decode(build([cmds], len(exp), 5, min_match=2, q_min=4, mutate=_patch(76, (5).to_bytes(4, "little"))))) == exp
    with pytest.raises(O.OracleError):
        O.decode(build([cmds], len(exp), 5, min_match=2, q_min=4, mutate=_patch(76, (6).to_bytes(4, "little"))))


def test_pair_symbols_follow_absolute_parity_and_fillers_are_dropped():
    # q_mode = 1 (FORMAT.md §1.7), q_min = 4, blocks of 32 bytes.  Block 0 is one LITQ run [0, 32): 16 full pairs.
    # Block 1: "p" [32] is LITA; copy(0, 2) -> [33, 35); the run "HIJKL" occupies [35, 40): pairs k = 17..19 =
    # (filler,H) (I,J) (K,L): 3 symbols for 5 bytes, the low half of pair 17 is position 34, outside the run;
    # copy(35, 2) -> [40, 42); "MNOPQ" occupies [42, 47): pairs 21..23 = (M,N) (O,P) (Q,filler);
    # copy(0, 2) -> [47, 49); "xyzw" occupies [49, 53): pairs 24..26 = (filler,x) (y,z) (w,filler): 3 symbols for 4 bytes.
    first = [(b"a" + bytes(range(98, 98 + 30)) + b"~", None)]
    blocks = [first, [(b"p", (0, 2)), (b"HIJKL", (35, 2)), (b"MNOPQ", (0, 2)), (b"xyzw", None)]]
    exp = first[0][0] + b"p" + b"ab" + b"HIJKL" + b"HI" + b"MNOPQ" + b"ab" + b"xyzw"
    outs = []
    for filler in (0x21, 0x7E, 0x00):
        a = build(blocks, len(exp), 5, min_match=2, q_min=4, q_mode=1, filler=filler)
        outs.append(bytes(O.decode(a)))
        s = O.segment(a, 1)
        assert (s["n_lit_a"], s["n_lit_q"], s["n_sym_q"]) == (1, 14, 9)
        assert s["out_pos"].tolist() == [32, 35, 42, 49] and s["lit_pos"].tolist() == [0, 0, 3, 6]
        assert O.segment(a, 0)["n_sym_q"] == 16
    assert outs == [exp] * 3 == [lz_reference(blocks, len(exp), 5)] * 3
    # the run "xyzw" ends at the odd position 53 = N: the filler half of its last pair lies past the end of the output
    import numpy as np
    canary = np.full(len(exp) + 8, 0xEE, dtype=np.uint8)
    assert bytes(O.decode_prefix(a, 2, check_levels=True, out=canary)) == exp and (canary[len(exp):] == 0xEE).all()
    h = O.header(a)
    assert h["q_mode"] == 1 and 1 <= h["n_qpairs"] <= 25
    # the pair table is sorted, strictly increasing: swapping two entries is rejected
    q = h["qtab_off"]
    e0, e1 = a[q:q + 4], a[q + 4:q + 8]
    with pytest.raises(O.OracleError):
        O.decode(build(blocks, len(exp), 5, min_match=2, q_min=4, q_mode=1, filler=0, mutate=_patch(q, e1 + e0)))


def test_self_overlap_seed_is_the_tail_of_the_own_literal_run_also_across_segments():
    # FORMAT.md §3 (c) with segments: "ab" ends segment 0 as a match-less command; segment 1 starts with copy(0, 6), whose
    # seed would be the literal run of ANOTHER command: rejected.  Restarted by its own literals it is legal.
    with pytest.raises(O.OracleError) as e:
        dec([[[(b"ab", None)], [(b"", (0, 6))]]], 8, 3, min_match=2)
    assert e.value.name == "E_CORRUPT"
    assert dec([[[(b"ab", None)], [(b"ab", (2, 4))]]], 8, 3, min_match=2) == b"abababab"
    # period 2 with a 3-byte run in front: the seed [1, 3) is the tail of the own run
    assert dec([[(b"xab", (1, 5))]], 8, 3, min_match=2) == b"xabababa"
