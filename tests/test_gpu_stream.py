"""-m gpu: the HBM-bound kernels (bs_lse_merge, bs_attn_bwd_prep, bs_attn_bwd_finish) through
the C-ABI against the fp64 oracle on the same seeded inputs."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from conftest import randn_bf16  # noqa: E402


def _imports():
    import torch
    from paper_2502_21231_b200 import binding as B
    import gpu_util as U
    return torch, B, U


@pytest.mark.parametrize("n,rows,Hq,D", [(1, 37, 4, 64), (2, 100, 6, 128), (8, 515, 16, 128),
                                          (64, 70, 48, 128), (5, 9, 3, 64),
                                          # n <= 4: several outputs per thread and pass; more heads
                                          # than one block owns (32), ragged last row tile
                                          (3, 61, 40, 128), (4, 131, 64, 64), (2, 9, 33, 128)])
def test_lse_merge_vs_oracle(nprng, n, rows, Hq, D):
    torch, B, U = _imports()
    O_bits = [randn_bf16(nprng, rows, Hq, D) for _ in range(n)]
    L = (3.0 * nprng.standard_normal((n, Hq, rows))).astype(np.float32)
    # sprinkle -inf parts, and make a few rows all -inf (no visible key anywhere)
    L[nprng.random((n, Hq, rows)) < 0.2] = -np.inf
    L[:, :, rows // 2] = -np.inf
    for s in range(n):  # parts with -inf LSE hold garbage that must be ignored
        bad = np.isneginf(L[s]).T
        O_bits[s][bad] = 0x7FC0  # NaN
    Od = [U.to_dev(b) for b in O_bits]
    Ld = [torch.from_numpy(L[s]).cuda() for s in range(n)]
    sh = B.make_shape(Hq, Hq, D, rows, rows)
    r0, r1 = (3, rows - 2) if rows > 20 else (0, rows)
    O_out = torch.full((rows, Hq, D), 7.0, dtype=torch.bfloat16, device="cuda")
    L_out = torch.full((Hq, rows), 7.0, dtype=torch.float32, device="cuda")
    B.lse_merge(Od, Ld, sh, (r0, r1), O_out, L_out)
    torch.cuda.synchronize()
    Of = np.stack([oracle.bf16_to_f64(b) for b in O_bits])
    Of[np.isnan(Of)] = 0.0
    Oo, Lo = oracle.merge(Of, L.astype(np.float64))
    got_O = oracle.bf16_to_f64(U.to_bits(O_out)).reshape(rows, Hq, D)
    got_L = L_out.double().cpu().numpy()
    # rows outside [r0,r1) untouched
    assert np.all(got_O[:r0] == 7.0) and np.all(got_O[r1:] == 7.0)
    assert np.all(got_L[:, :r0] == 7.0) and np.all(got_L[:, r1:] == 7.0)
    got_O, got_L, Oo, Lo = got_O[r0:r1], got_L[:, r0:r1], Oo[r0:r1], Lo[:, r0:r1]
    assert np.array_equal(np.isneginf(got_L), np.isneginf(Lo))
    fin = np.isfinite(Lo)
    assert np.abs(got_L[fin] - Lo[fin]).max() <= 1e-4
    # one bf16 output rounding (2^-9 relative) + fp32 noise
    assert np.all(np.abs(got_O - Oo) <= 2.0 ** -8 * np.abs(Oo) + 1e-5)
    # running merge: output aliases part 0
    B.lse_merge(Od, Ld, sh, (0, rows), Od[0], Ld[0])
    torch.cuda.synchronize()
    a = oracle.bf16_to_f64(U.to_bits(Od[0])).reshape(rows, Hq, D)[r0:r1]
    assert np.array_equal(a, got_O)


@pytest.mark.parametrize("rows,Hq,D", [(33, 4, 64), (200, 6, 128), (1000, 32, 128)])
def test_bwd_prep_and_finish(nprng, rows, Hq, D):
    torch, B, U = _imports()
    O_bits, dO_bits = randn_bf16(nprng, rows, Hq, D), randn_bf16(nprng, rows, Hq, D)
    O, dO = U.to_dev(O_bits), U.to_dev(dO_bits)
    sh = B.make_shape(Hq, Hq, D, rows, rows)
    delta = torch.full((Hq, rows), float("nan"), dtype=torch.float32, device="cuda")
    acc = torch.full((rows, Hq, D), float("nan"), dtype=torch.float32, device="cuda")
    B.attn_bwd_prep(sh, O, dO, delta, acc)
    torch.cuda.synchronize()
    want = np.einsum("ihd,ihd->hi", oracle.bf16_to_f64(O_bits), oracle.bf16_to_f64(dO_bits))
    assert np.abs(delta.double().cpu().numpy() - want).max() <= 1e-4
    assert torch.all(acc == 0)
    x = torch.from_numpy(nprng.standard_normal((rows, Hq, D)).astype(np.float32)).cuda()
    dQ = torch.empty((rows, Hq, D), dtype=torch.bfloat16, device="cuda")
    B.attn_bwd_finish(sh, x, dQ)
    torch.cuda.synchronize()
    from conftest import f32_to_bf16_bits
    assert np.array_equal(U.to_bits(dQ), f32_to_bf16_bits(x.cpu().numpy()))


def test_reduce_probe_leaves_the_accumulator_unchanged():
    """bs_reduce_probe (measurement aid): fp32 reduce-add boxes of zeros into dQ_acc-shaped memory."""
    import torch
    from paper_2502_21231_b200 import binding as B
    g = torch.Generator(device="cuda").manual_seed(3)
    acc = torch.randn((1024, 3, 128), generator=g, device="cuda", dtype=torch.float32)
    acc[5, 1, 7] = float("inf")
    want = acc.clone()
    B.reduce_probe(acc, 64)
    B.reduce_probe(acc, 0)
    torch.cuda.synchronize()
    assert torch.equal(acc.view(torch.int32), want.view(torch.int32))
    with pytest.raises(B.BsError):
        B.reduce_probe(torch.zeros((100, 3, 128), device="cuda"), 4)       # rows not a multiple of 128
    with pytest.raises(B.BsError):
        B.reduce_probe(torch.zeros((128, 3, 48), device="cuda"), 4)        # head_dim not a multiple of 32
