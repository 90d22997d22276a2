"""-m gpu: the parts of the C-ABI contract the workload tests do not reach: padded row strides, a
padded LSE head stride, an explicit softmax scale, an output row sub-range (rows outside it are
not written), a call with no segments at all, and the argument errors that must be reported
before any launch (include/bytescale_attn.h)."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from conftest import randn_bf16  # noqa: E402
from paper_2502_21231_b200 import binding as B  # noqa: E402


def _dev(bits):
    import gpu_util as U
    return U.to_dev(bits)


def test_strides_scale_and_row_subrange(nprng):
    import gpu_util as U
    Hq, Hkv, D, rows = 4, 2, 128, 700
    qs, ks = Hq * D + 64, Hkv * D + 8          # padded row strides (multiples of 8 elements)
    lse_stride = rows + 24
    scale = 0.05
    # documents: [0,300) and [300,700); the call owns output rows [300,700) only
    seqs = [(300, 1, 0), (400, 1, 0)]
    pl = B.plan(seqs)
    segs = [s for s in pl["steps"][0]["segs"] if s[0] >= 300]
    assert len(segs) == 1
    Qb, Kb, Vb, dOb = (randn_bf16(nprng, rows, H, D) for H in (Hq, Hkv, Hkv, Hq))

    def padded(bits, H, stride):
        buf = torch.full((rows, stride), float("nan"), dtype=torch.bfloat16, device="cuda")
        buf[:, :H * D] = _dev(bits).view(rows, H * D)
        return buf
    Q, K, V, dO = padded(Qb, Hq, qs), padded(Kb, Hkv, ks), padded(Vb, Hkv, ks), padded(dOb, Hq, qs)
    O = torch.full((rows, qs), 7.0, dtype=torch.bfloat16, device="cuda")
    LSE = torch.full((Hq, lse_stride), 7.0, dtype=torch.float32, device="cuda")
    sh = B.make_shape(Hq, Hkv, D, rows, rows, softmax_scale=scale, q_row_stride=qs, kv_row_stride=ks,
                      lse_head_stride=lse_stride)
    ws = torch.empty(B.attn_workspace_bytes(sh, len(segs), False), dtype=torch.uint8, device="cuda")
    B.attn_fwd(sh, Q, K, V, segs, (300, rows), O, LSE, ws)
    torch.cuda.synchronize()
    # rows outside the range, the stride padding and the LSE padding are untouched
    assert torch.all(O[:300] == 7.0) and torch.all(O[:, Hq * D:] == 7.0)
    assert torch.all(LSE[:, :300] == 7.0) and torch.all(LSE[:, rows:] == 7.0)
    q_seq = np.concatenate([np.zeros(300, np.int32), np.ones(400, np.int32)])
    q_pos = np.concatenate([np.arange(300), np.arange(400)]).astype(np.int32)
    sel = np.arange(300, rows)
    Oo, Lo = oracle.attn_fwd(Qb[sel], Kb, Vb, q_seq[sel], q_pos[sel], q_seq, q_pos, scale=scale)
    got_O = oracle.bf16_to_f64(U.to_bits(O[300:, :Hq * D].contiguous())).reshape(400, Hq, D)
    got_L = LSE[:, 300:rows].double().cpu().numpy()
    assert np.abs(got_O - Oo).max() <= U.TOL_O
    assert np.abs(got_L - Lo).max() <= U.TOL_LSE
    # backward with the same strides: dK/dV rows of the uncovered document are zero
    delta = torch.empty((Hq, lse_stride), dtype=torch.float32, device="cuda")
    acc = torch.empty((rows, Hq, D), dtype=torch.float32, device="cuda")
    B.attn_bwd_prep(sh, O, dO, delta, acc)
    dK = torch.full((rows, ks), float("nan"), dtype=torch.bfloat16, device="cuda")
    dV = torch.full((rows, ks), float("nan"), dtype=torch.bfloat16, device="cuda")
    wsb = torch.empty(B.attn_workspace_bytes(sh, len(segs), True), dtype=torch.uint8, device="cuda")
    B.attn_bwd(sh, Q, K, V, dO, LSE, delta, segs, acc, dK, dV, wsb)
    dQ = torch.full((rows, qs), 7.0, dtype=torch.bfloat16, device="cuda")
    B.attn_bwd_finish(sh, acc, dQ)
    torch.cuda.synchronize()
    dQo, dKo, dVo = oracle.attn_bwd(Qb[sel], Kb, Vb, dOb[sel], q_seq[sel], q_pos[sel], q_seq, q_pos,
                                    scale=scale)
    g_dQ = oracle.bf16_to_f64(U.to_bits(dQ[300:, :Hq * D].contiguous())).reshape(400, Hq, D)
    g_dK = oracle.bf16_to_f64(U.to_bits(dK[:, :Hkv * D].contiguous())).reshape(rows, Hkv, D)
    g_dV = oracle.bf16_to_f64(U.to_bits(dV[:, :Hkv * D].contiguous())).reshape(rows, Hkv, D)
    assert U.rel_l2(g_dQ, dQo) <= U.TOL_GRAD
    assert U.rel_l2(g_dK, dKo) <= U.TOL_GRAD and U.rel_l2(g_dV, dVo) <= U.TOL_GRAD
    assert np.all(g_dK[:300] == 0) and np.all(g_dV[:300] == 0)
    assert np.all(oracle.bf16_to_f64(U.to_bits(dQ[:300, :Hq * D].contiguous())) == 0)  # acc was 0 there
    assert torch.all(dQ[:, Hq * D:] == 7.0)


def test_no_segments_fills_the_range():
    Hq, Hkv, D, rows = 2, 1, 64, 50
    sh = B.make_shape(Hq, Hkv, D, rows, rows)
    z = torch.zeros((rows, Hq, D), dtype=torch.bfloat16, device="cuda")
    kv = torch.zeros((rows, Hkv, D), dtype=torch.bfloat16, device="cuda")
    O = torch.full((rows, Hq, D), 3.0, dtype=torch.bfloat16, device="cuda")
    LSE = torch.full((Hq, rows), 3.0, dtype=torch.float32, device="cuda")
    ws = torch.empty(B.attn_workspace_bytes(sh, 0, False), dtype=torch.uint8, device="cuda")
    B.attn_fwd(sh, z, kv, kv, [], (10, 40), O, LSE, ws)
    torch.cuda.synchronize()
    assert torch.all(O[10:40] == 0) and torch.all(torch.isneginf(LSE[:, 10:40]))
    assert torch.all(O[:10] == 3.0) and torch.all(O[40:] == 3.0) and torch.all(LSE[:, :10] == 3.0)


def test_argument_errors_are_reported_before_any_launch():
    Hq, Hkv, D, rows = 2, 1, 64, 300
    sh = B.make_shape(Hq, Hkv, D, rows, rows)
    q = torch.zeros((rows, Hq, D), dtype=torch.bfloat16, device="cuda")
    kv = torch.zeros((rows, Hkv, D), dtype=torch.bfloat16, device="cuda")
    O = torch.full((rows, Hq, D), 3.0, dtype=torch.bfloat16, device="cuda")
    LSE = torch.full((Hq, rows), 3.0, dtype=torch.float32, device="cuda")
    ws = torch.empty(B.attn_workspace_bytes(sh, 2, False), dtype=torch.uint8, device="cuda")
    bad = [
        [(0, 200, 0, 200, 0, 0), (100, 300, 0, 300, 0, 0)],   # q ranges overlap without being identical
        [(0, 400, 0, 300, 0, 0)],                             # q range outside the buffer
        [(0, 100, 200, 100, 0, 0)],                           # empty / reversed k range
    ]
    for segs in bad:
        with pytest.raises(B.BsError) as e:
            B.attn_fwd(sh, q, kv, kv, segs, (0, rows), O, LSE, ws)
        assert e.value.code == -1
    with pytest.raises(B.BsError) as e:   # workspace too small
        B.attn_fwd(sh, q, kv, kv, [(0, 300, 0, 300, 0, 0)], (0, rows), O, LSE, ws[:64])
    assert e.value.code == -3
    with pytest.raises(B.BsError) as e:   # head_dim 96 is not supported
        B.attn_workspace_bytes(B.make_shape(2, 1, 96, rows, rows), 1, False)
    assert e.value.code == -2
    torch.cuda.synchronize()
    assert torch.all(O == 3.0) and torch.all(LSE == 3.0)    # nothing was launched


def _fwd_bwd(sh, Q, K, V, dO, segs, rows_q, rows_k):
    """One forward + backward of a single call; returns O, LSE, dQ, dK, dV (device tensors)."""
    Hq, Hkv, D = sh.n_q_heads, sh.n_kv_heads, sh.head_dim
    O = torch.full((rows_q, Hq, D), float("nan"), dtype=torch.bfloat16, device="cuda")
    LSE = torch.full((Hq, rows_q), float("nan"), dtype=torch.float32, device="cuda")
    ws = torch.empty(B.attn_workspace_bytes(sh, len(segs), False), dtype=torch.uint8, device="cuda")
    B.attn_fwd(sh, Q, K, V, segs, (0, rows_q), O, LSE, ws)
    delta = torch.empty((Hq, rows_q), dtype=torch.float32, device="cuda")
    acc = torch.empty((rows_q, Hq, D), dtype=torch.float32, device="cuda")
    B.attn_bwd_prep(sh, O, dO, delta, acc)
    dK = torch.full((rows_k, Hkv, D), float("nan"), dtype=torch.bfloat16, device="cuda")
    dV = torch.full((rows_k, Hkv, D), float("nan"), dtype=torch.bfloat16, device="cuda")
    wsb = torch.empty(B.attn_workspace_bytes(sh, len(segs), True), dtype=torch.uint8, device="cuda")
    B.attn_bwd(sh, Q, K, V, dO, LSE, delta, segs, acc, dK, dV, wsb)
    dQ = torch.empty((rows_q, Hq, D), dtype=torch.bfloat16, device="cuda")
    B.attn_bwd_finish(sh, acc, dQ)
    torch.cuda.synchronize()
    return O, LSE, dQ, dK, dV


def _same(a_list, b_list, what):
    """O, LSE, dK, dV bit for bit; dQ (index 2) to one bf16 ulp: its fp32 partial sums are added
    in L2 in whatever order the key tiles finish."""
    for i, (a, b) in enumerate(zip(a_list, b_list)):
        if i == 2:
            assert torch.allclose(a.float(), b.float(), rtol=2.0 ** -7, atol=1e-6), what
        else:
            assert torch.equal(a.view(torch.uint8), b.view(torch.uint8)), what


def test_causal_offset_sentinels(nprng):
    """causal_offset = INT32_MAX ("every key") and INT32_MIN ("no key") are legal: the library
    stores offsets clamped to [-q_len, k_len], which leaves the mask unchanged, so the kernels'
    32-bit row + offset arithmetic cannot overflow (a mismatch between the host's and the device's
    block counts would hang the kernel)."""
    Hq, Hkv, D, rq, rk = 4, 2, 128, 300, 500
    Qb, dOb = randn_bf16(nprng, rq, Hq, D), randn_bf16(nprng, rq, Hq, D)
    Kb, Vb = randn_bf16(nprng, rk, Hkv, D), randn_bf16(nprng, rk, Hkv, D)
    Q, K, V, dO = _dev(Qb), _dev(Kb), _dev(Vb), _dev(dOb)
    sh = B.make_shape(Hq, Hkv, D, rq, rk)
    ref = _fwd_bwd(sh, Q, K, V, dO, [(0, rq, 0, rk, rk - 1, 0)], rq, rk)
    for off in (2 ** 31 - 1, 2 ** 30, rk + 5):
        _same(ref, _fwd_bwd(sh, Q, K, V, dO, [(0, rq, 0, rk, off, 0)], rq, rk), off)
    for off in (-2 ** 31, -2 ** 30, -rq):
        O, LSE, dQ, dK, dV = _fwd_bwd(sh, Q, K, V, dO, [(0, rq, 0, rk, off, 0)], rq, rk)
        assert torch.all(O == 0) and torch.all(torch.isneginf(LSE))
        assert torch.all(dQ == 0) and torch.all(dK == 0) and torch.all(dV == 0)
    # two segments on one query range, one with a sentinel offset: softmax over the union
    segs = [(0, rq, 0, 200, 2 ** 31 - 1, 0), (0, rq, 200, rk, -40, 0)]
    same = [(0, rq, 0, 200, 199, 0), (0, rq, 200, rk, -40, 0)]
    _same(_fwd_bwd(sh, Q, K, V, dO, segs, rq, rk), _fwd_bwd(sh, Q, K, V, dO, same, rq, rk), "union")


@pytest.mark.parametrize("Hq,Hkv,D", [(4, 2, 128), (2, 2, 64)])
def test_nan_in_rows_no_segment_covers(nprng, Hq, Hkv, D):
    """Fixed-capacity or torch.empty-padded buffers: rows that no segment covers may hold anything,
    NaN and Inf included.  TMA loads whole 128-row boxes, so such rows sit in shared memory right
    behind a ragged range end; masked P is 0, and 0 x NaN must not reach any covered row's O, dQ,
    dK or dV.  Ranges of 333 and 70 rows (ragged in every tile), garbage rows between and after."""
    import gpu_util as U
    cap = 600
    docs = [(0, 333), (400, 470)]   # [begin, end) rows of the two documents in every buffer
    bad = float("nan")

    def buf(bits, H, fill):
        t = torch.full((cap, H, D), fill, dtype=torch.bfloat16, device="cuda")
        for i, (a, b) in enumerate(docs):
            t[a:b] = _dev(bits[i]).view(b - a, H, D)
        return t
    Qb = [randn_bf16(nprng, b - a, Hq, D) for a, b in docs]
    dOb = [randn_bf16(nprng, b - a, Hq, D) for a, b in docs]
    Kb = [randn_bf16(nprng, b - a, Hkv, D) for a, b in docs]
    Vb = [randn_bf16(nprng, b - a, Hkv, D) for a, b in docs]
    sh = B.make_shape(Hq, Hkv, D, cap, cap)
    segs = [(a, b, a, b, 0, i) for i, (a, b) in enumerate(docs)]
    outs = {}
    for fill in (0.0, bad, float("inf")):
        Q, dO, K, V = buf(Qb, Hq, fill), buf(dOb, Hq, fill), buf(Kb, Hkv, fill), buf(Vb, Hkv, fill)
        outs[fill if fill == fill else "nan"] = _fwd_bwd(sh, Q, K, V, dO, segs, cap, cap)
    # rows no segment covers: O = 0, LSE = -inf, dK = dV = 0, whatever they held
    for key, (O, LSE, dQ, dK, dV) in outs.items():
        for t in (O, dQ, dK, dV):
            assert not torch.isnan(t.float()).any(), f"NaN with fill {key}"
        assert torch.all(O[333:400] == 0) and torch.all(O[470:] == 0)
        assert torch.all(torch.isneginf(LSE[:, 333:400])) and torch.all(torch.isneginf(LSE[:, 470:]))
        assert torch.all(dK[333:400] == 0) and torch.all(dV[470:] == 0)
    # and the covered rows do not depend on the garbage at all
    for key in ("nan", float("inf")):
        _same(outs[0.0], outs[key], f"fill {key} changed a result")
    # against the oracle
    q_seq = np.concatenate([np.full(b - a, i, np.int32) for i, (a, b) in enumerate(docs)])
    q_pos = np.concatenate([np.arange(b - a, dtype=np.int32) for a, b in docs])
    cat = lambda xs: np.concatenate(xs)  # noqa: E731
    Oo, Lo = oracle.attn_fwd(cat(Qb), cat(Kb), cat(Vb), q_seq, q_pos, q_seq, q_pos)
    O, LSE, dQ, dK, dV = outs["nan"]
    rows = torch.cat([torch.arange(a, b) for a, b in docs]).cuda()
    f64 = lambda t, H: oracle.bf16_to_f64(U.to_bits(t[rows].contiguous())).reshape(len(rows), H, D)  # noqa: E731
    got_O, got_L = f64(O, Hq), LSE[:, rows].double().cpu().numpy()
    U.o_compare(got_O, Oo, "NaN-padded buffers: ")
    assert np.abs(got_L - Lo).max() <= U.TOL_LSE
    dl = np.ascontiguousarray((got_O * oracle.bf16_to_f64(cat(dOb))).sum(-1).T)
    for strict, kw in ((False, {}), (True, dict(LSE=got_L, delta=dl))):
        ref = oracle.attn_bwd(cat(Qb), cat(Kb), cat(Vb), cat(dOb), q_seq, q_pos, q_seq, q_pos, **kw)
        for name, g, want in zip(("dQ", "dK", "dV"), (f64(dQ, Hq), f64(dK, Hkv), f64(dV, Hkv)), ref):
            U.grad_compare(name, g, want, q_seq, "NaN-padded buffers: ", strict)
