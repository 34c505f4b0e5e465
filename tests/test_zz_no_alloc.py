"""af_argmax_rows_static (include/af.h): the ArgMax of Alg. 1 l.5/l.8 with its scratch in a static __device__
array, for callers that cannot allocate.  It must return exactly the tokens of the existing path, af_argmax_rows (an
integer decided on the stored fp32 logits by an order-free rule: bit-exact, the tolerance of every index test here),
on two calls in a row (the array keeps the first call's contents), and refuse sizes beyond its maximum.

Collected last on purpose (the file name sorts after every other test file): the suite runs with `pytest -x`.
It stands alone - no fixture or state of another test file - so it passes in a fresh process and after the others.
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

MAX_ROWS = 256   # AF_ARGMAX_STATIC_MAX_ROWS


def _logits(n_rows, vocab, seed):
    g = torch.Generator().manual_seed(seed)
    x = torch.randn(n_rows, vocab, generator=g, dtype=torch.float32)
    if n_rows >= 4 and vocab >= 64:
        x[0, 7] = x[0, vocab - 3] = 50.0            # a tie across chunks: the lowest index wins
        x[1, :] = 0.25                              # every entry equal -> 0
        x[2, :] = float("nan")                      # only NaNs -> 0
        x[3, vocab // 2] = float("nan")             # NaNs are never selected
        x[3, vocab - 1] = 60.0                      # the maximum in the ragged last chunk
    return x.cuda()


@pytest.mark.parametrize("n_rows,vocab", [(9, 151936), (1, 152064), (256, 4099), (5, 100), (33, 2048 * 64 + 1)])
def test_static_argmax_equals_existing_path_twice_in_a_row(n_rows, vocab):
    from paper_2512_20276_b200 import binding as B
    a, b = _logits(n_rows, vocab, 11), _logits(n_rows, vocab, 12)
    ref_a, ref_b = B.argmax_rows(a), B.argmax_rows(b)
    out = torch.full((n_rows,), -7, dtype=torch.int32, device="cuda")
    B.argmax_rows_static(a, out)
    got_a = out.clone()
    B.argmax_rows_static(b, out)                    # second call: the scratch still holds the first call's candidates
    got_b = out.clone()
    torch.cuda.synchronize()
    assert torch.equal(got_a, ref_a) and torch.equal(got_b, ref_b)
    # and both agree with the definition, written out on the host (lowest index of the maximum, NaNs never selected)
    for x, got in ((a, got_a), (b, got_b)):
        xn = x.cpu().numpy()
        want = np.argmax(np.where(np.isnan(xn), -np.inf, xn), axis=1)   # numpy: first occurrence of the maximum
        want[np.all(np.isnan(xn), axis=1)] = 0
        assert np.array_equal(got.cpu().numpy(), want.astype(np.int32))


def test_static_argmax_rejects_more_rows_than_its_scratch_holds_and_allocates_nothing():
    from paper_2512_20276_b200 import binding as B
    x = _logits(MAX_ROWS + 1, 128, 3)
    out = torch.full((MAX_ROWS + 1,), -7, dtype=torch.int32, device="cuda")
    with pytest.raises(Exception) as e:
        B.argmax_rows_static(x, out)
    assert "static scratch" in str(e.value)
    torch.cuda.synchronize()
    assert int((out != -7).sum()) == 0              # nothing was enqueued
    # no device memory is taken by a call (cudaMemGetInfo: driver-level free bytes; one call first, so that the
    # driver's lazy load of the kernel's code is not counted)
    y = _logits(MAX_ROWS, 4099, 5)
    o2 = torch.empty(MAX_ROWS, dtype=torch.int32, device="cuda")
    B.argmax_rows_static(y, o2)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        B.argmax_rows_static(y, o2)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0
    assert torch.equal(o2, B.argmax_rows(y))
