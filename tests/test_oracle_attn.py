"""Pins of the fp64 oracle (oracle/oracle_attn.c) against things other than itself:
brute-force dense masked softmax, closed forms, invariances, finite differences, identities.
CPU only."""
import numpy as np
import pytest

import oracle
from conftest import f32_to_bf16_bits, randn_bf16

F = oracle.bf16_to_f64


def packed_rows(lens):
    seq = np.concatenate([np.full(L, i, np.int32) for i, L in enumerate(lens)])
    pos = np.concatenate([np.arange(L, dtype=np.int32) for L in lens])
    return seq, pos


def brute_force(Q, K, V, q_seq, q_pos, k_seq, k_pos, scale):
    """Dense T x T masked softmax with an explicit mask matrix (independent of the oracle)."""
    Qf, Kf, Vf = F(Q), F(K), F(V)
    nq, Hq, D = Qf.shape
    nk, Hkv, _ = Kf.shape
    G = Hq // Hkv
    mask = (q_seq[:, None] == k_seq[None, :]) & (k_pos[None, :] <= q_pos[:, None])
    O = np.zeros((nq, Hq, D))
    LSE = np.full((Hq, nq), -np.inf)
    for h in range(Hq):
        S = scale * Qf[:, h, :] @ Kf[:, h // G, :].T
        E = np.where(mask, np.exp(S - np.where(mask, S, -np.inf).max(axis=1, initial=-1e300,
                                                                    keepdims=True)), 0.0)
        rs = E.sum(axis=1)
        ok = rs > 0
        mx = np.where(mask, S, -np.inf).max(axis=1, initial=-1e300)
        LSE[h, ok] = mx[ok] + np.log(rs[ok])
        P = np.zeros_like(E)
        P[ok] = E[ok] / rs[ok, None]
        O[:, h, :] = P @ Vf[:, h // G, :]
    return O, LSE


@pytest.mark.parametrize("Hq,Hkv,D", [(2, 2, 8), (4, 2, 16), (6, 1, 8)])
def test_fwd_vs_brute_force(nprng, Hq, Hkv, D):
    lens = [1, 5, 17, 2, 30]
    seq, pos = packed_rows(lens)
    T = len(seq)
    Q, K, V = randn_bf16(nprng, T, Hq, D), randn_bf16(nprng, T, Hkv, D), randn_bf16(nprng, T, Hkv, D)
    scale = 1.0 / np.sqrt(D)
    O, LSE = oracle.attn_fwd(Q, K, V, seq, pos, seq, pos, scale)
    Ob, Lb = brute_force(Q, K, V, seq, pos, seq, pos, scale)
    np.testing.assert_allclose(O, Ob, rtol=0, atol=1e-13)
    np.testing.assert_allclose(LSE, Lb, rtol=0, atol=1e-13)


def test_fwd_brute_force_partial_keys_and_empty_rows(nprng):
    # queries at global positions 3..8 of seq 0, keys = positions 5..12 -> rows 3,4 see nothing
    Hq, Hkv, D = 4, 2, 8
    q_pos = np.arange(3, 9, dtype=np.int32)
    k_pos = np.arange(5, 13, dtype=np.int32)
    q_seq = np.zeros(6, np.int32)
    k_seq = np.zeros(8, np.int32)
    Q, K, V = randn_bf16(nprng, 6, Hq, D), randn_bf16(nprng, 8, Hkv, D), randn_bf16(nprng, 8, Hkv, D)
    O, LSE = oracle.attn_fwd(Q, K, V, q_seq, q_pos, k_seq, k_pos, 0.3)
    Ob, Lb = brute_force(Q, K, V, q_seq, q_pos, k_seq, k_pos, 0.3)
    np.testing.assert_allclose(O, Ob, atol=1e-13)
    assert np.all(np.isneginf(LSE[:, :2])) and np.all(O[:2] == 0)
    np.testing.assert_allclose(LSE[:, 2:], Lb[:, 2:], atol=1e-13)


def test_closed_forms_forward(nprng):
    Hq, Hkv, D = 4, 2, 16
    G = Hq // Hkv
    lens = [1, 9, 1, 23]
    seq, pos = packed_rows(lens)
    T = len(seq)
    Q, K, V = randn_bf16(nprng, T, Hq, D), randn_bf16(nprng, T, Hkv, D), randn_bf16(nprng, T, Hkv, D)
    scale = 0.25
    O, LSE = oracle.attn_fwd(Q, K, V, seq, pos, seq, pos, scale)
    Qf, Kf, Vf = F(Q), F(K), F(V)
    first = np.flatnonzero(pos == 0)
    for i in first:  # row 0 of every document (incl. length-1 documents): O = its V row
        for h in range(Hq):
            np.testing.assert_allclose(O[i, h], Vf[i, h // G], atol=1e-15)
            np.testing.assert_allclose(LSE[h, i], scale * Qf[i, h] @ Kf[i, h // G], atol=1e-14)
    # V constant over a document => O = that constant, for any Q, K
    Vc = np.zeros((T, Hkv, D), np.float32)
    consts = nprng.standard_normal((len(lens), Hkv, D)).astype(np.float32)
    Vc[:] = consts[seq]
    Vc = f32_to_bf16_bits(Vc)
    Oc, _ = oracle.attn_fwd(Q, K, Vc, seq, pos, seq, pos, scale)
    np.testing.assert_allclose(Oc, np.repeat(F(Vc), G, axis=1), atol=1e-14)
    # Q = 0 => LSE = ln(pos+1), O = prefix mean of V within the document
    Q0 = np.zeros_like(Q)
    O0, L0 = oracle.attn_fwd(Q0, K, V, seq, pos, seq, pos, scale)
    np.testing.assert_allclose(L0, np.broadcast_to(np.log(pos + 1.0), (Hq, T)), atol=1e-14)
    for i in range(T):
        start = i - pos[i]
        pm = Vf[start:i + 1].mean(axis=0)
        np.testing.assert_allclose(O0[i], np.repeat(pm, G, axis=0), atol=1e-14)


def test_packing_order_invariance(nprng):
    Hq, Hkv, D = 2, 1, 8
    lens = [7, 1, 12, 4]
    seq, pos = packed_rows(lens)
    T = len(seq)
    Q, K, V = randn_bf16(nprng, T, Hq, D), randn_bf16(nprng, T, Hkv, D), randn_bf16(nprng, T, Hkv, D)
    dO = randn_bf16(nprng, T, Hq, D)
    O, LSE = oracle.attn_fwd(Q, K, V, seq, pos, seq, pos)
    g = oracle.attn_bwd(Q, K, V, dO, seq, pos, seq, pos)
    # permute whole documents (and, since rows carry (seq,pos), even arbitrary rows)
    perm = nprng.permutation(T)
    O2, LSE2 = oracle.attn_fwd(Q[perm], K[perm], V[perm], seq[perm], pos[perm], seq[perm], pos[perm])
    g2 = oracle.attn_bwd(Q[perm], K[perm], V[perm], dO[perm], seq[perm], pos[perm], seq[perm],
                         pos[perm])
    np.testing.assert_allclose(O2, O[perm], atol=1e-14)
    np.testing.assert_allclose(LSE2, LSE[:, perm], atol=1e-14)
    for a, b in zip(g2, g):
        np.testing.assert_allclose(a, b[perm], atol=1e-13)


def _objective(Q, K, V, dO, seq, pos, scale):
    """sum(O * dO) evaluated by the dense brute force in fp64 on fp64 inputs."""
    nq, Hq, D = Q.shape
    G = Hq // K.shape[1]
    mask = (seq[:, None] == seq[None, :]) & (pos[None, :] <= pos[:, None])
    tot = 0.0
    for h in range(Hq):
        S = scale * Q[:, h] @ K[:, h // G].T
        S = np.where(mask, S, -np.inf)
        P = np.exp(S - S.max(axis=1, keepdims=True))
        P /= P.sum(axis=1, keepdims=True)
        tot += np.sum((P @ V[:, h // G]) * dO[:, h])
    return tot


def test_bwd_finite_differences(nprng):
    Hq, Hkv, D = 4, 2, 4
    lens = [3, 6, 1]
    seq, pos = packed_rows(lens)
    T = len(seq)
    Q, K, V = randn_bf16(nprng, T, Hq, D), randn_bf16(nprng, T, Hkv, D), randn_bf16(nprng, T, Hkv, D)
    dO = randn_bf16(nprng, T, Hq, D)
    scale = 0.5
    dQ, dK, dV = oracle.attn_bwd(Q, K, V, dO, seq, pos, seq, pos, scale)
    base = [F(Q), F(K), F(V)]
    dOf = F(dO)
    eps = 1e-6
    for idx, grad in enumerate((dQ, dK, dV)):
        num = np.zeros_like(grad)
        it = np.nditer(grad, flags=["multi_index"])
        for _ in it:
            mi = it.multi_index
            args_p = [a.copy() for a in base]
            args_m = [a.copy() for a in base]
            args_p[idx][mi] += eps
            args_m[idx][mi] -= eps
            num[mi] = (_objective(*args_p, dOf, seq, pos, scale) -
                       _objective(*args_m, dOf, seq, pos, scale)) / (2 * eps)
        np.testing.assert_allclose(grad, num, rtol=0, atol=2e-7)


def test_bwd_identities_and_closed_forms(nprng):
    Hq, Hkv, D = 4, 2, 8
    G = Hq // Hkv
    lens = [1, 11, 19]
    seq, pos = packed_rows(lens)
    T = len(seq)
    Q, K, V = randn_bf16(nprng, T, Hq, D), randn_bf16(nprng, T, Hkv, D), randn_bf16(nprng, T, Hkv, D)
    dO = randn_bf16(nprng, T, Hq, D)
    scale = 0.3
    dQ, dK, dV = oracle.attn_bwd(Q, K, V, dO, seq, pos, seq, pos, scale)
    Qf, Kf, Vf, dOf = F(Q), F(K), F(V), F(dO)
    for doc in range(len(lens)):
        rows = np.flatnonzero(seq == doc)
        # softmax shift invariance: sum_j dK_j = 0 per document and kv head
        np.testing.assert_allclose(dK[rows].sum(axis=0), 0, atol=1e-13)
        # rows of P sum to 1: sum_j dV_j = sum_{h in g} sum_i dO_i
        want = dOf[rows].sum(axis=0).reshape(Hkv, G, D).sum(axis=1)
        np.testing.assert_allclose(dV[rows].sum(axis=0), want, atol=1e-13)
        # Q <- tQ, K <- K/t invariance: sum_i q_i.dq_i (over group) = sum_j k_j.dk_j
        lhs = (Qf[rows] * dQ[rows]).reshape(len(rows), Hkv, G, D).sum(axis=(0, 2, 3))
        rhs = (Kf[rows] * dK[rows]).sum(axis=(0, 2))
        np.testing.assert_allclose(lhs, rhs, atol=1e-12)
    # row 0 of any document: dQ = 0; length-1 document: dK = 0, dV = sum_group dO
    first = np.flatnonzero(pos == 0)
    np.testing.assert_allclose(dQ[first], 0, atol=1e-15)
    np.testing.assert_allclose(dK[0], 0, atol=1e-15)
    np.testing.assert_allclose(dV[0], dOf[0].reshape(Hkv, G, D).sum(axis=1), atol=1e-15)
    # Q = 0: dK = 0 and dV_j = sum_{i >= j, same doc} dO_i / (pos_i + 1)
    Q0 = np.zeros_like(Q)
    dQ0, dK0, dV0 = oracle.attn_bwd(Q0, K, V, dO, seq, pos, seq, pos, scale)
    np.testing.assert_allclose(dK0, 0, atol=1e-15)
    for j in range(T):
        later = np.flatnonzero((seq == seq[j]) & (pos >= pos[j]))
        want = (dOf[later] / (pos[later] + 1.0)[:, None, None]).sum(axis=0)
        np.testing.assert_allclose(dV0[j], want.reshape(Hkv, G, D).sum(axis=1), atol=1e-14)
    # K = 0 => dQ = 0
    dQk, _, _ = oracle.attn_bwd(Q, np.zeros_like(K), V, dO, seq, pos, seq, pos, scale)
    np.testing.assert_allclose(dQk, 0, atol=1e-15)


@pytest.mark.parametrize("L,N", [(64, 4), (50, 4), (7, 4), (96, 3), (5, 8)])
def test_chunk_and_merge_invariance(nprng, L, N):
    """Zigzag-sharded, per-step partial attention merged over the ring == unsharded attention,
    for every rank; backward with merged LSE/delta sums to the full backward."""
    Hq, Hkv, D = 2, 1, 8
    G = Hq // Hkv
    Qg, Kg, Vg = randn_bf16(nprng, L, Hq, D), randn_bf16(nprng, L, Hkv, D), randn_bf16(nprng, L, Hkv, D)
    dOg = randn_bf16(nprng, L, Hq, D)
    seq0, posg = np.zeros(L, np.int32), np.arange(L, dtype=np.int32)
    O_full, LSE_full = oracle.attn_fwd(Qg, Kg, Vg, seq0, posg, seq0, posg)
    dQ_full, dK_full, dV_full = oracle.attn_bwd(Qg, Kg, Vg, dOg, seq0, posg, seq0, posg)
    dK_sum = np.zeros_like(dK_full)
    dV_sum = np.zeros_like(dV_full)
    for r in range(N):
        pl = oracle.oracle_plan([(L, N, r)])
        qs, qp = oracle.rows_from_plan(pl)
        if len(qp) == 0:
            continue
        Q, dO = Qg[qp], dOg[qp]
        Os, Ls = [], []
        for s in range(N):
            ks, kp = oracle.rows_from_plan(pl, s)
            O_s, L_s = oracle.attn_fwd(Q, Kg[kp], Vg[kp], qs, qp, ks, kp)
            Os.append(O_s)
            Ls.append(L_s)
        O_m, L_m = oracle.merge(np.stack(Os), np.stack(Ls))
        np.testing.assert_allclose(O_m, O_full[qp], atol=1e-13)
        np.testing.assert_allclose(L_m, LSE_full[:, qp], atol=1e-13)
        delta = np.einsum("ihd,ihd->hi", F(dO), O_m)
        dQ_acc = np.zeros((len(qp), Hq, D))
        for s in range(N):
            ks, kp = oracle.rows_from_plan(pl, s)
            dq, dk, dv = oracle.attn_bwd(Q, Kg[kp], Vg[kp], dO, qs, qp, ks, kp, LSE=L_m, delta=delta)
            dQ_acc += dq
            np.add.at(dK_sum, kp, dk)
            np.add.at(dV_sum, kp, dv)
        np.testing.assert_allclose(dQ_acc, dQ_full[qp], atol=1e-13)
    # Eq. 1 == Eq. 2: summed over ranks the contributions are the gradient
    np.testing.assert_allclose(dK_sum, dK_full, atol=1e-12)
    np.testing.assert_allclose(dV_sum, dV_full, atol=1e-12)


def test_merge_special_cases(nprng):
    rows, Hq, D = 5, 3, 4
    O1 = nprng.standard_normal((rows, Hq, D))
    L1 = nprng.standard_normal((Hq, rows))
    # n = 1 is the identity
    O, L = oracle.merge(O1[None], L1[None])
    np.testing.assert_allclose(O, O1, atol=1e-15)
    np.testing.assert_allclose(L, L1, atol=1e-15)
    # a part with LSE = -inf is ignored even if its O is garbage
    junk = np.full((rows, Hq, D), np.nan)
    O, L = oracle.merge(np.stack([O1, junk]), np.stack([L1, np.full((Hq, rows), -np.inf)]))
    np.testing.assert_allclose(O, O1, atol=1e-15)
    np.testing.assert_allclose(L, L1, atol=1e-15)
    # all -inf -> (0, -inf), never NaN
    ninf = np.full((Hq, rows), -np.inf)
    O, L = oracle.merge(np.stack([O1, O1]), np.stack([ninf, ninf]))
    assert np.all(O == 0) and np.all(np.isneginf(L))
    # two equal-LSE parts average; closed form ln 2 shift
    O2 = nprng.standard_normal((rows, Hq, D))
    O, L = oracle.merge(np.stack([O1, O2]), np.stack([L1, L1]))
    np.testing.assert_allclose(O, 0.5 * (O1 + O2), atol=1e-15)
    np.testing.assert_allclose(L, L1 + np.log(2.0), atol=1e-15)
    # n-way == iterated pairwise
    Os = nprng.standard_normal((4, rows, Hq, D))
    Ls = 3 * nprng.standard_normal((4, Hq, rows))
    O, L = oracle.merge(Os, Ls)
    Oi, Li = Os[0], Ls[0]
    for s in range(1, 4):
        Oi, Li = oracle.merge(np.stack([Oi, Os[s]]), np.stack([Li, Ls[s]]))
    np.testing.assert_allclose(O, Oi, atol=1e-14)
    np.testing.assert_allclose(L, Li, atol=1e-14)
    # direct definition in numpy (logsumexp / weighted mean)
    w = np.exp(Ls - Ls.max(axis=0))
    w /= w.sum(axis=0)
    np.testing.assert_allclose(L, np.log(np.exp(Ls).sum(axis=0)), atol=1e-13)
    np.testing.assert_allclose(O, np.einsum("shi,sihd->ihd", w, Os), atol=1e-14)
