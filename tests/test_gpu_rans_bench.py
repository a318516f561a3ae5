"""The entropy stage alone ("256 MB exponential, batch 4096 x 64 KB"): the GPU rANS row
encoder and decoder against the oracle's plain C row coder (oracle/acx_rans_rows.c), word for word."""
import numpy as np
import pytest
import torch

from acx_build import normalise
from oracle import acx_rans_rows as R

pytestmark = pytest.mark.gpu


def exponential_rows(n_rows, row_bytes, seed=6, scale=12.0):
    rng = np.random.default_rng(seed)
    return np.minimum(rng.exponential(scale=scale, size=(n_rows, row_bytes)), 255).astype(np.uint8)


@pytest.mark.parametrize("n_rows,row_bytes", [(1, 1), (3, 31), (5, 33), (7, 1000), (300, 4096), (64, 65536), (9, 70001)])
def test_rows_bit_exact_vs_oracle(n_rows, row_bytes):
    from paper_2606_18900_b200.aceapex import RansBatch
    rows = exponential_rows(n_rows, row_bytes, seed=n_rows)
    freq = normalise(np.bincount(rows.ravel(), minlength=256).tolist())
    want_enc, want_sizes = R.encode(rows, freq)
    rb = RansBatch(freq, row_bytes)
    assert rb.row_cap == want_enc.shape[1]
    d_rows = torch.from_numpy(rows).cuda()
    enc, sizes = rb.encode(d_rows)
    torch.cuda.synchronize()
    got_sizes = sizes.cpu().numpy().astype(np.uint32)
    assert np.array_equal(got_sizes, want_sizes)
    got = enc[:n_rows * rb.row_cap].cpu().numpy().reshape(n_rows, rb.row_cap)
    for r in range(n_rows):                                   # heads and words, byte for byte (the slack behind a row is unspecified)
        assert np.array_equal(got[r, :got_sizes[r]], want_enc[r, :want_sizes[r]]), r
    out = rb.decode(enc, sizes, n_rows)
    assert rb.status() == 0
    assert np.array_equal(out.cpu().numpy(), rows)
    # the oracle's decoder reads the GPU's rows, and the GPU decoder reads the oracle's rows
    assert np.array_equal(R.decode(got, got_sizes, row_bytes, freq), rows)
    enc2 = torch.zeros(n_rows * rb.row_cap + 128, dtype=torch.uint8, device="cuda")
    enc2[:n_rows * rb.row_cap] = torch.from_numpy(want_enc.ravel()).cuda()
    out2 = rb.decode(enc2, torch.from_numpy(want_sizes.astype(np.int32)).cuda(), n_rows)
    assert rb.status() == 0 and np.array_equal(out2.cpu().numpy(), rows)


def test_skewed_tables_and_corruption():
    from paper_2606_18900_b200.aceapex import RansBatch
    rng = np.random.default_rng(1)
    for probs in ([1.0], [0.999, 0.001], [0.5, 0.25, 0.125, 0.125]):
        rows = rng.choice(len(probs), size=(40, 5000), p=probs).astype(np.uint8) + 65
        freq = normalise(np.bincount(rows.ravel(), minlength=256).tolist())
        want_enc, want_sizes = R.encode(rows, freq)
        rb = RansBatch(freq, 5000)
        enc, sizes = rb.encode(torch.from_numpy(rows).cuda())
        torch.cuda.synchronize()
        assert np.array_equal(sizes.cpu().numpy().astype(np.uint32), want_sizes)
        assert np.array_equal(rb.decode(enc, sizes, 40).cpu().numpy(), rows) and rb.status() == 0
    enc[3 * rb.row_cap + 5] ^= 0x10                         # a flipped bit in a row's head: the final-state check sees it
    rb.decode(enc, sizes, 40)
    assert rb.status() == 1


def test_the_papers_batch_shape():
    """4096 rows of 64 KB (256 MiB): encode -> decode identity on the device, sampled rows word for word against the oracle."""
    from paper_2606_18900_b200.aceapex import RansBatch
    rows = exponential_rows(4096, 65536)
    freq = normalise(np.bincount(rows.ravel(), minlength=256).tolist())
    rb = RansBatch(freq, 65536)
    d_rows = torch.from_numpy(rows).cuda()
    enc, sizes = rb.encode(d_rows)
    out = rb.decode(enc, sizes, 4096)
    assert rb.status() == 0 and torch.equal(out, d_rows)
    pick = np.array([0, 1, 77, 2048, 4095])
    want_enc, want_sizes = R.encode(rows[pick], freq)
    got_sizes = sizes.cpu().numpy().astype(np.uint32)
    for k, r in enumerate(pick):
        assert got_sizes[r] == want_sizes[k]
        assert np.array_equal(enc[r * rb.row_cap:r * rb.row_cap + int(got_sizes[r])].cpu().numpy(), want_enc[k, :want_sizes[k]])
