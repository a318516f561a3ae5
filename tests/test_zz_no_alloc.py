"""aceapex_rans_encode_static (include/aceapex.h): the rANS row encoder for callers that may not allocate (scratch in a
file-scope static __device__ array of the library) against the existing aceapex_rans_encode, bit for bit (the bar of the
other GPU tests: byte and index work is exact), on two calls in a row that share the static array.  Collected last on
purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _rows(n_rows, row_bytes, seed):
    rng = np.random.default_rng(seed)
    return np.minimum(rng.exponential(scale=12.0, size=(n_rows, row_bytes)), 255).astype(np.uint8)


def _freq(rows):
    hist = np.bincount(rows.ravel(), minlength=256).astype(np.int64)
    freq = np.maximum((hist * 2048) // hist.sum(), (hist > 0).astype(np.int64))      # 2^11 slots, every present symbol >= 1
    while freq.sum() != 2048:
        freq[int(np.argmax(freq))] += 1 if freq.sum() < 2048 else -1
    return freq.astype(np.uint16)


def _same(rb, a, b, n_rows):
    (enc_a, sizes_a), (enc_b, sizes_b) = a, b
    torch.cuda.synchronize()
    sa, sb = sizes_a.cpu().numpy(), sizes_b.cpu().numpy()
    assert np.array_equal(sa, sb)
    ea = enc_a[:n_rows * rb.row_cap].cpu().numpy().reshape(n_rows, rb.row_cap)
    eb = enc_b[:n_rows * rb.row_cap].cpu().numpy().reshape(n_rows, rb.row_cap)
    for r in range(n_rows):                                   # heads and words; the slack behind a row is unspecified
        assert np.array_equal(ea[r, :sa[r]], eb[r, :sb[r]]), r


@pytest.mark.parametrize("n_rows,row_bytes", [(300, 4097), (5000, 1000), (600, 65536), (1, 1)])
def test_static_scratch_encoder_matches_the_existing_path_twice(n_rows, row_bytes):
    from paper_2606_18900_b200.aceapex import RansBatch, load
    assert load().aceapex_rans_static_setup() == 0
    first, second = _rows(n_rows, row_bytes, 1), _rows(n_rows, row_bytes, 2)
    rb = RansBatch(_freq(np.concatenate([first, second])), row_bytes)
    for rows in (first, second):                              # the second call finds the first call's words in the array
        d = torch.from_numpy(rows).cuda()
        want = rb.encode(d)
        got = rb.encode_static(d)
        _same(rb, want, got, n_rows)
        out = rb.decode(got[0], got[1], n_rows)
        assert rb.status() == 0 and np.array_equal(out.cpu().numpy(), rows)


def test_static_scratch_encoder_rejects_rows_beyond_its_maximum():
    from paper_2606_18900_b200.aceapex import AceapexError, RansBatch
    rows = _rows(2, 65537, 3)
    rb = RansBatch(_freq(rows), 65537)
    d = torch.from_numpy(rows).cuda()
    rb.encode(d)                                              # the existing path takes it
    with pytest.raises(AceapexError) as e:
        rb.encode_static(d)
    assert e.value.name == "E_TOO_LARGE"
    torch.cuda.synchronize()
