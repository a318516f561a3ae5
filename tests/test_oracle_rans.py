"""Pins of the oracle's rANS step (FORMAT.md §1.7) against an independent pure-Python encoder (tests/acx_build.py),
closed forms and the final-state invariant."""
import math

import numpy as np
import pytest

from acx_build import M, MQ_BITS, normalise, rans_encode
from oracle import acx_oracle as O


def roundtrip(symbols, tids, freqs):
    states, streams = rans_encode(list(symbols), list(tids), freqs)
    sym, final, used = O.rans_decode(np.array(freqs, dtype=np.uint16), np.array(tids, dtype=np.uint8),
                                     np.array(states, dtype=np.uint32), streams)
    assert used.tolist() == [len(s) for s in streams]   # every state consumed exactly its own stream
    assert (final == (1 << 16)).all()               # encoder started at 2^16 -> decoder ends there
    assert list(sym) == list(symbols)
    return states, [w for s in streams for w in s]


@pytest.mark.parametrize("n", [0, 1, 31, 32, 33, 64, 1000])
def test_identity_random(n):
    rng = np.random.default_rng(n)
    s = rng.integers(0, 256, n)
    hist = np.bincount(s, minlength=256).tolist()
    roundtrip(s.tolist(), [0] * n, [normalise(hist)])


def test_single_symbol_alphabet_needs_no_words():
    f = [0] * 256
    f[65] = M
    states, words = roundtrip([65] * 500, [0] * 500, [f])
    assert words == [] and states == [1 << 16] * 32     # x = M * (x >> 11) + (x & (M-1)) is the identity


def test_two_symbols_freq_1_and_M_minus_1():
    f = [0] * 256
    f[0], f[1] = 1, M - 1
    rng = np.random.default_rng(7)
    s = (rng.random(5000) < 0.999).astype(int)
    s[::700] = 0
    roundtrip(s.tolist(), [0] * len(s), [f])


def test_worked_example_by_hand():
    # One symbol 'a' (freq 512, cum 0 in a table {a:512, b:1536}) on state 0, encoder side by hand:
    #   x = 2^16 = 65536; f << 21 = 2^30 > x -> no word; x' = (65536 // 512) << 11 + 65536 % 512 + 0 = 128 * 2048 = 262144
    # Decoder: slot = 262144 & 2047 = 0 -> 'a'; x = 512 * (262144 >> 11) + 0 - 0 = 65536.
    f = [0] * 256
    f[97], f[98] = 512, 1536
    states, streams = rans_encode([97], [0], [f])
    assert states[0] == 262144 and states[1:] == [65536] * 31 and streams == [[]] * 32
    sym, final, used = O.rans_decode(np.array([f], np.uint16), np.array([0], np.uint8), np.array(states, np.uint32), streams)
    assert list(sym) == [97] and final[0] == 65536 and used.sum() == 0
    # 'b' (freq 1536, cum 512): x' = (65536 // 1536) << 11 + 65536 % 1536 + 512 = 42 * 2048 + 1024 + 512 = 87552
    states, streams = rans_encode([98], [0], [f])
    assert states[0] == 87552 and streams == [[]] * 32
    sym, final, used = O.rans_decode(np.array([f], np.uint16), np.array([0], np.uint8), np.array(states, np.uint32), streams)
    assert list(sym) == [98] and final[0] == 65536


def test_closed_form_size():
    # compressed bits = sum -log2(f_s / M) + 32 x 16 bits of initial-state slack, within a small additive slack
    rng = np.random.default_rng(11)
    p = np.array([0.5, 0.25, 0.125, 0.0625, 0.0625])
    s = rng.choice(5, size=20000, p=p)
    f = [0] * 256
    for k, q in enumerate(p):
        f[k] = int(q * M)
    states, words = roundtrip(s.tolist(), [0] * len(s), [f])
    ideal = sum(-math.log2(f[v] / M) for v in s)
    bits = 16 * len(words) + sum(math.log2(x) - 16 for x in states)
    assert abs(bits - ideal) < 64            # rANS loses far less than one bit per state here


def test_several_tables_interleaved_on_the_same_states():
    rng = np.random.default_rng(3)
    a = rng.integers(0, 4, 333)
    b = rng.integers(100, 256, 777)
    s = np.concatenate([a, b])
    t = [0] * len(a) + [1] * len(b)
    fa = normalise(np.bincount(a, minlength=256).tolist())
    fb = normalise(np.bincount(b, minlength=256).tolist())
    roundtrip(s.tolist(), t, [fa, fb])


def test_worked_example_with_words_on_two_states():
    # Table {a: 1, b: 2047}.  Decoding by hand, FORMAT.md §1.5, symbols i = 0, 1, 32 (states 0, 1, 0):
    #   state 0 starts at x = 65536 * 2048 + 0 = 134217728: slot 0 -> 'a' (cum 0, freq 1); x = 1 * (x >> 11) + 0 = 65536.
    #   state 1 starts at 65537 * 2048 = 134219776: slot 0 -> 'a'; x = 65537.
    #   i = 32 (state 0): x = 65536: slot 0 -> 'a'; x = 1 * 32 + 0 = 32 < 2^16 -> x = (32 << 16) | w with w from state 0's stream.
    # Choose w0 = 0x1234 for state 0 and give state 1 a different word 0xBEEF that must NOT be touched:
    f = [0] * 256
    f[97], f[98] = 1, 2047
    streams = [[0x1234], [0xBEEF]] + [[] for _ in range(30)]
    states = [134217728, 134219776] + [65536] * 30
    tids = [0] * 33
    # symbols 2..31 are decoded on states 2..31 = 65536: slot 0 -> 'a', x = 32 -> needs a word: give each a stream of one word
    for k in range(2, 32):
        streams[k] = [k]
    sym, final, used = O.rans_decode(np.array([f], np.uint16), np.array(tids, np.uint8), np.array(states, np.uint32), streams)
    assert list(sym) == [97] * 33
    assert final[0] == (32 << 16) | 0x1234          # state 0 read its own word, after its second symbol
    assert final[1] == 65537                         # state 1 never renormalised
    assert [int(final[k]) for k in range(2, 32)] == [(32 << 16) | k for k in range(2, 32)]
    assert used.tolist() == [1, 0] + [1] * 30


def test_states_do_not_share_words():
    # the same symbols coded twice; swapping two states' streams must change the output (streams are per state)
    rng = np.random.default_rng(9)
    s = rng.integers(0, 256, 2000)
    f = normalise(np.bincount(s, minlength=256).tolist())
    states, streams = rans_encode(s.tolist(), [0] * len(s), [f])
    assert streams[3] != streams[4]
    swapped = list(streams)
    swapped[3], swapped[4] = streams[4], streams[3]
    try:
        sym, final, used = O.rans_decode(np.array([f], np.uint16), np.zeros(len(s), np.uint8), np.array(states, np.uint32), swapped)
        assert list(sym) != s.tolist()
    except O.OracleError as e:
        assert e.name == "E_TRUNCATED"


def test_truncated_word_stream_is_an_error():
    rng = np.random.default_rng(5)
    s = rng.integers(0, 256, 400)
    f = normalise(np.bincount(s, minlength=256).tolist())
    states, streams = rans_encode(s.tolist(), [0] * 400, [f])
    k = max(range(32), key=lambda q: len(streams[q]))
    streams[k] = streams[k][:-1]                       # one state's stream is one word short
    with pytest.raises(O.OracleError) as e:
        O.rans_decode(np.array([f], np.uint16), np.zeros(400, np.uint8), np.array(states, np.uint32), streams)
    assert e.value.name == "E_TRUNCATED"


def test_worked_example_pair_table_precision_12():
    # FORMAT.md §1.7: the pair table codes with pb = 12 (M_Q = 4096).  Two entries {A: 1024, B: 3072}, by hand:
    #   encode A on x = 65536: f << 20 = 2^30 > x -> no word; x' = (65536 // 1024) << 12 + 0 + 0 = 64 * 4096 = 262144
    #   decode: slot = 262144 & 4095 = 0 -> A; x = 1024 * (262144 >> 12) + 0 = 65536.
    #   encode B: x' = (65536 // 3072) << 12 + 65536 % 3072 + 1024 = 21 * 4096 + 1024 + 1024 = 88064
    #   decode: slot = 88064 & 4095 = 2048 -> B (cum 1024); x = 3072 * 21 + 2048 - 1024 = 65536.
    f = [1024, 3072]
    for sym, want in ((0, 262144), (1, 88064)):
        states, streams = rans_encode([sym], [0], [f], [MQ_BITS])
        assert states[0] == want and states[1:] == [65536] * 31 and streams == [[]] * 32
        got, final, used = O.rans_decode(np.array([f], np.uint16), np.array([0], np.uint8), np.array(states, np.uint32), streams,
                                         prob_bits=MQ_BITS)
        assert list(got) == [sym] and final[0] == 65536 and used.sum() == 0
    # the same states read with pb = 11 are a different code: 262144 & 2047 = 0 still says A but leaves x = 512 * 128 != 2^16
    with pytest.raises(O.OracleError):
        O.rans_decode(np.array([f], np.uint16), np.array([0], np.uint8), np.array([262144] + [65536] * 31, np.uint32), [[]] * 32, prob_bits=11)


def test_tables_of_precision_11_and_12_interleaved_on_the_same_states():
    # a segment's symbol sequence ends with LITA (pb 11) followed by LITQ pairs (pb 12, up to 4096 symbols) on the SAME 32 states
    rng = np.random.default_rng(21)
    a = rng.integers(0, 40, 1237)                                   # byte symbols
    b = rng.integers(0, 900, 2999)                                  # pair-table entries
    n_sym = 900
    fa = normalise(np.bincount(a, minlength=n_sym).tolist())        # sums to 2^11
    fb = normalise(np.bincount(b, minlength=n_sym).tolist(), MQ_BITS)
    syms = a.tolist() + b.tolist()
    tids = [0] * len(a) + [1] * len(b)
    states, streams = rans_encode(syms, tids, [fa, fb], [11, MQ_BITS])
    got, final, used = O.rans_decode(np.array([fa, fb], np.uint16), np.array(tids, np.uint8), np.array(states, np.uint32), streams,
                                     prob_bits=[11, MQ_BITS])
    assert list(got) == syms and (final == 65536).all() and used.tolist() == [len(s) for s in streams]
    ideal = sum(-math.log2(fa[v] / 2048) for v in a) + sum(-math.log2(fb[v] / 4096) for v in b)
    bits = 16 * sum(len(s) for s in streams) + sum(math.log2(x) - 16 for x in states)
    assert abs(bits - ideal) < 64


# ---- the row coder of the entropy micro-benchmark (oracle/acx_rans_rows.c) ----------------

def exponential_rows(n_rows, row_bytes, seed=6, scale=12.0):
    """The micro-benchmark's data shape: exponentially distributed byte values ("256 MB exponential")."""
    rng = np.random.default_rng(seed)
    return np.minimum(rng.exponential(scale=scale, size=(n_rows, row_bytes)), 255).astype(np.uint8)


@pytest.mark.parametrize("row_bytes", [1, 31, 32, 33, 1000, 4096])
def test_row_encoder_matches_the_python_encoder_word_for_word(row_bytes):
    from oracle import acx_rans_rows as R
    rows = exponential_rows(3, row_bytes, seed=row_bytes)
    freq = normalise(np.bincount(rows.ravel(), minlength=256).tolist())
    enc, sizes = R.encode(rows, freq)
    for r in range(rows.shape[0]):
        states, streams = rans_encode(rows[r].tolist(), [0] * row_bytes, [freq])
        words = [w for st in streams for w in st]
        assert sizes[r] == 256 + 2 * len(words)
        head = np.frombuffer(enc[r, :256].tobytes(), dtype="<u4").reshape(32, 2)
        assert head[:, 0].tolist() == states
        assert head[:, 1].tolist() == np.concatenate([[0], np.cumsum([len(st) for st in streams])[:-1]]).tolist()
        assert np.frombuffer(enc[r, 256:sizes[r]].tobytes(), dtype="<u2").tolist() == words
        # and the oracle's own decoder (FORMAT.md 1.7) reads it back
        sym, final, used = O.rans_decode(np.array([freq], np.uint16), np.zeros(row_bytes, np.uint8), np.array(states, np.uint32), streams)
        assert sym.tolist() == rows[r].tolist() and (final == 65536).all()
    assert np.array_equal(R.decode(enc, sizes, row_bytes, freq), rows)


def test_row_coder_size_is_the_entropy_bound():
    from oracle import acx_rans_rows as R
    rows = exponential_rows(8, 65536)
    freq = normalise(np.bincount(rows.ravel(), minlength=256).tolist())
    enc, sizes = R.encode(rows, freq)
    ideal_bits = sum(-math.log2(freq[v] / M) for v in rows.ravel())
    got_bits = 8 * (int(sizes.sum()) - 256 * 8)                       # payload words only
    assert abs(got_bits - ideal_bits) < 8 * 32 * 32 + 0.001 * ideal_bits   # at most ~one word per state and row, 0.1 % slack
    assert np.array_equal(R.decode(enc, sizes, 65536, freq), rows)
    bad = enc.copy()
    bad[3, 300] ^= 0x40
    with pytest.raises(ValueError):
        R.decode(bad, sizes, 65536, freq)
