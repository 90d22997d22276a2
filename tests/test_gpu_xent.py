"""-m gpu: bs_softmax_xent (fused softmax cross-entropy) against the fp64 oracle,
element by element: several vocabulary sizes (rows that fit shared memory and rows that do not,
a ragged tail of vocab % 8 logits, a padded row stride), ignored tokens, large-magnitude logits.
Tolerances: loss in fp32 over up to 128K terms - 2e-5 absolute + 2e-6 relative; dlogits is
rounded to bf16 once (2^-9 relative) after fp32 arithmetic - 2^-8 relative + 1e-7 absolute."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

from oracle.xent import softmax_xent as oracle_xent  # noqa: E402
from paper_2502_21231_b200 import binding as B  # noqa: E402


def run(T, V, stride, scale, std, seed, ignore_every=0):
    g = torch.Generator().manual_seed(seed)
    x = (torch.randn(T, stride, generator=g) * std).bfloat16()
    y = torch.randint(0, V, (T,), generator=g, dtype=torch.int32)
    if ignore_every:
        y[::ignore_every] = -100
    xd, yd = x.cuda(), y.cuda()
    loss = torch.full((T,), 7.0, dtype=torch.float32, device="cuda")
    d = torch.full((T, stride), 7.0, dtype=torch.bfloat16, device="cuda")
    B.softmax_xent(xd, yd, scale, loss, d, vocab=V)
    torch.cuda.synchronize()
    lo, do = oracle_xent(x[:, :V].double().numpy(), y.numpy(), scale)
    got_l, got_d = loss.double().cpu().numpy(), d.double().cpu().numpy()
    assert np.all(np.abs(got_l - lo) <= 2e-5 + 2e-6 * np.abs(lo)), np.abs(got_l - lo).max()
    err = np.abs(got_d[:, :V] - do)
    assert np.all(err <= 2.0 ** -8 * np.abs(do) + 1e-7), err.max()
    if stride > V:
        assert np.all(got_d[:, V:] == 7.0)      # the stride padding is not written


@pytest.mark.parametrize("V", [8, 1000, 1003, 16384, 49152, 50264, 131072])
def test_against_oracle(V):
    stride = (V + 7) // 8 * 8
    run(37 if V < 100000 else 9, V, stride, 1.0 / 37, 3.0, V)


def test_padded_stride_ignored_tokens_and_large_logits():
    run(64, 4096, 4096 + 64, 0.25, 1.0, 1, ignore_every=5)
    run(16, 2048, 2048, 1.0, 30.0, 2)           # |x| up to ~120: exp underflow / max handling


def test_argument_errors():
    x = torch.zeros(4, 24, dtype=torch.bfloat16, device="cuda")
    y = torch.zeros(4, dtype=torch.int32, device="cuda")
    loss = torch.zeros(4, device="cuda")
    call = B.lib.bs_softmax_xent
    assert call(x.data_ptr(), y.data_ptr(), 4, 24, 20, 1.0, loss.data_ptr(), x.data_ptr(), None) == -1
    assert call(x.data_ptr(), y.data_ptr(), 4, 20, 20, 1.0, loss.data_ptr(), x.data_ptr(), None) == -1
    assert call(None, y.data_ptr(), 4, 24, 24, 1.0, loss.data_ptr(), x.data_ptr(), None) == -1
    assert call(None, None, 0, 24, 24, 1.0, None, None, None) == 0      # empty call
