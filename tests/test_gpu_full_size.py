"""-m gpu: BASELINE.json configs 2-5 at FULL size through the C-ABI, in the launch configuration
bench.py uses (one bs_attn_fwd / bs_attn_bwd per ring step over the whole buffer, the first
forward clearing dQ_acc, bs_lse_merge over all steps, prep / finish once).

A full fp64 oracle pass is hours at these sizes, so the comparison is
  * cfg2: four whole heads (MHA heads are independent) - every element of O, LSE, dQ, dK, dV of
    those heads over all 32768 rows against the oracle;
  * O, LSE and dQ of a seeded sample of query rows (first / last row of every part, rows next to
    128-row tile boundaries, random rows), each against the oracle over ALL keys of the sequence -
    these outputs depend on their own row only, so the sample is exact;
  * sparse-dO run: the backward again, same launches, with dO non-zero only on
    a sampled row set R.  Then dK and dV of EVERY key row (and dQ of R) are exactly what the
    oracle computes from the rows of R alone, at cost |R| x keys: every element of dK / dV of
    every KV head is compared, per 128-key tile of every ring step, and dQ outside R must be 0
    (oracle formulas under the LSE and delta the kernel was given, see gpu_util.grad_compare);
  * dense dO: dK, dV of every key row through the O(T) identities that hold for any set of query
    rows (softmax rows sum to 1, softmax shift invariance):
        sum_j dV[j,g,:] = sum_{h in g} sum_i dO[i,h,:]        sum_j dK[j,g,:] = 0      per sequence
    and  sum_i Q_i . dQ_i (heads of g) = sum_j K_j . dK_j      per sequence and KV group.
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

import oracle  # noqa: E402
from paper_2502_21231_b200 import binding as B  # noqa: E402
from paper_2502_21231_b200.synth import rng, workloads  # noqa: E402


def _sample_rows(pl, n_random, seed, n_boundary=24):
    """Local Q rows to check: part boundaries, tile boundaries, a few random ones."""
    cu = pl["cu_rows_q"]
    rows = set()
    for a, b in zip(cu[:-1], cu[1:]):
        if b > a:
            rows.update([a, b - 1])
            mid = (a + b) // 2  # for a zigzag shard this is where the high part starts
            rows.update(x for x in (mid - 1, mid, a + 127, a + 128) if a <= x < b)
        if len(rows) >= n_boundary:
            break
    rows = set(sorted(rows)[:n_boundary])
    g = np.random.default_rng(seed)
    rows.update(int(x) for x in g.integers(0, pl["q_rows"], n_random))
    return np.array(sorted(rows), np.int64)


class FullRun:
    """One config at full size on the device; keeps what the checks need."""

    def __init__(self, cfg):
        import gpu_util as U
        self.U, self.cfg = U, cfg
        w = self.w = workloads.make_workload(cfg)
        self.Hq, self.Hkv, self.D = w.n_q_heads, w.n_kv_heads, w.head_dim
        Hq, Hkv, D = self.Hq, self.Hkv, self.D
        pl = self.pl = B.plan(w.seqs)
        self.opl = oracle.oracle_plan(w.seqs)
        self.rows_q, self.n_steps = pl["q_rows"], pl["n_steps"]
        qruns = workloads.runs_from(pl["q_seq"], pl["q_pos"])
        self.Qb = workloads.gen_rows(w.seed, rng.STREAM_Q, qruns, Hq * D)
        self.dOb = workloads.gen_rows(w.seed, rng.STREAM_DO, qruns, Hq * D)
        self.Q = U.to_dev(self.Qb).view(self.rows_q, Hq, D)
        self.dO = U.to_dev(self.dOb).view(self.rows_q, Hq, D)
        self.acc = torch.full((self.rows_q, Hq, D), float("nan"), dtype=torch.float32, device="cuda")
        self.Kb, self.Vb, self.Kd, self.Vd = [], [], [], []
        for s in range(self.n_steps):
            st = pl["steps"][s]
            kruns = workloads.runs_from(st["k_seq"], st["k_pos"])
            self.Kb.append(workloads.gen_rows(w.seed, rng.STREAM_K, kruns, Hkv * D))
            self.Vb.append(workloads.gen_rows(w.seed, rng.STREAM_V, kruns, Hkv * D))
            self.Kd.append(U.to_dev(self.Kb[-1]).view(-1, Hkv, D))
            self.Vd.append(U.to_dev(self.Vb[-1]).view(-1, Hkv, D))
        self.sh0 = B.make_shape(Hq, Hkv, D, self.rows_q, pl["steps"][0]["kv_rows"])

    def forward(self):
        Hq, Hkv, D, rows_q = self.Hq, self.Hkv, self.D, self.rows_q
        parts = []
        for s in range(self.n_steps):
            st = self.pl["steps"][s]
            sh = B.make_shape(Hq, Hkv, D, rows_q, st["kv_rows"])
            O = torch.empty((rows_q, Hq, D), dtype=torch.bfloat16, device="cuda")
            L = torch.empty((Hq, rows_q), dtype=torch.float32, device="cuda")
            ws = torch.empty(B.attn_workspace_bytes(sh, len(st["segs"]), False), dtype=torch.uint8,
                             device="cuda")
            # as in bench.py: the first step's forward also clears the fp32 dQ accumulator
            B.attn_fwd(sh, self.Q, self.Kd[s], self.Vd[s], st["segs"], (0, rows_q), O, L, ws,
                       self.acc if s == 0 else None)
            parts.append((O, L))
        if self.n_steps > 1:
            self.O = torch.empty_like(parts[0][0])
            self.LSE = torch.empty_like(parts[0][1])
            B.lse_merge([p[0] for p in parts], [p[1] for p in parts], self.sh0, (0, rows_q), self.O,
                        self.LSE)
        else:
            self.O, self.LSE = parts[0]
        torch.cuda.synchronize()

    def backward(self, dO, clear_in_prep):
        """prep, every ring step's bs_attn_bwd, finish -> dQ, [dK per step], [dV per step]."""
        Hq, Hkv, D, rows_q = self.Hq, self.Hkv, self.D, self.rows_q
        delta = torch.empty((Hq, rows_q), dtype=torch.float32, device="cuda")
        B.attn_bwd_prep(self.sh0, self.O, dO, delta, self.acc if clear_in_prep else None)
        dKs, dVs = [], []
        for s in range(self.n_steps):
            st = self.pl["steps"][s]
            sh = B.make_shape(Hq, Hkv, D, rows_q, st["kv_rows"])
            dK = torch.full_like(self.Kd[s], float("nan"))
            dV = torch.full_like(self.Vd[s], float("nan"))
            ws = torch.empty(B.attn_workspace_bytes(sh, len(st["segs"]), True), dtype=torch.uint8,
                             device="cuda")
            B.attn_bwd(sh, self.Q, self.Kd[s], self.Vd[s], dO, self.LSE, delta, st["segs"], self.acc,
                       dK, dV, ws)
            dKs.append(dK)
            dVs.append(dV)
        dQ = torch.empty_like(self.Q)
        B.attn_bwd_finish(self.sh0, self.acc, dQ)
        torch.cuda.synchronize()
        return dQ, dKs, dVs

    # ------------------------------------------------------------------ oracle-side pieces
    def key_meta(self):
        ks = np.concatenate([self.opl["steps"][s]["k_seq"] for s in range(self.n_steps)])
        kp = np.concatenate([self.opl["steps"][s]["k_pos"] for s in range(self.n_steps)])
        return ks, kp

    def kv_heads(self, bits_list, heads):
        """bf16 bits [all keys of all steps, len(heads), D] of the given KV heads."""
        return np.concatenate([b.reshape(-1, self.Hkv, self.D)[:, heads] for b in bits_list])

    def key_blocks(self):
        """Block id per key row of the concatenated steps: (step, document, 128-row chunk)."""
        out, base = [], 0
        for s in range(self.n_steps):
            b = self.U._blocks(0, self.opl["steps"][s]["k_seq"], len(self.w.seqs)) + base
            base = int(b.max()) + 1
            out.append(b)
        return np.concatenate(out)

    def bits_of(self, t):
        return oracle.bf16_to_f64(self.U.to_bits(t.contiguous()))


def _check_sampled_rows(fr, dQ, n_random, n_boundary):
    U, cfg, Hq, Hkv, D, rows_q = fr.U, fr.cfg, fr.Hq, fr.Hkv, fr.D, fr.rows_q
    rows = _sample_rows(fr.pl, n_random, fr.w.seed, n_boundary)
    ks, kp = fr.key_meta()
    Kall = np.concatenate(fr.Kb).reshape(-1, Hkv, D)
    Vall = np.concatenate(fr.Vb).reshape(-1, Hkv, D)
    qs, qp = fr.opl["q_seq"][rows], fr.opl["q_pos"][rows]
    Qs, dOs = fr.Qb.reshape(rows_q, Hq, D)[rows], fr.dOb.reshape(rows_q, Hq, D)[rows]
    ridx = torch.from_numpy(rows).cuda()
    got_O = fr.bits_of(fr.O[ridx]).reshape(len(rows), Hq, D)
    got_L = fr.LSE[:, ridx].double().cpu().numpy()
    got_dQ = fr.bits_of(dQ[ridx]).reshape(len(rows), Hq, D)
    Oo, Lo = oracle.attn_fwd(Qs, Kall, Vall, qs, qp, ks, kp)
    dQo, _, _ = oracle.attn_bwd(Qs, Kall, Vall, dOs, qs, qp, ks, kp)
    # the same rows under the LSE and delta the backward kernel was given (gpu_util.grad_compare)
    dl = np.ascontiguousarray((got_O * oracle.bf16_to_f64(dOs)).sum(-1).T)
    dQi, _, _ = oracle.attn_bwd(Qs, Kall, Vall, dOs, qs, qp, ks, kp, LSE=got_L, delta=dl)
    del Kall, Vall
    label = f"cfg{cfg} ({len(rows)} sampled rows): "
    U.o_compare(got_O, Oo, label)
    err_L = float(np.abs(got_L - Lo).max())
    assert err_L <= U.TOL_LSE, f"cfg{cfg}: LSE abs err {err_L}"
    # every sampled row is its own block: dQ of a row depends on that row only
    U.grad_compare("dQ", got_dQ, dQo, np.arange(len(rows)), label, strict=False)
    U.grad_compare("dQ", got_dQ, dQi, np.arange(len(rows)), label, strict=True)
    print(f"{label}LSE abs err {err_L:.1e}")


def _check_identities(fr, dQ, dKs, dVs):
    cfg, Hq, Hkv, D, rows_q, pl = fr.cfg, fr.Hq, fr.Hkv, fr.D, fr.rows_q, fr.pl
    G = Hq // Hkv
    n_seq = len(fr.w.seqs)
    qseq = torch.from_numpy(np.ascontiguousarray(pl["q_seq"]).astype(np.int64)).cuda()
    sum_dO = torch.zeros((n_seq, Hkv, D), dtype=torch.float64, device="cuda")
    sum_dO.index_add_(0, qseq, fr.dO.double().view(rows_q, Hkv, G, D).sum(2))
    q_dq = torch.zeros((n_seq, Hkv), dtype=torch.float64, device="cuda")
    q_dq.index_add_(0, qseq, (fr.Q.double() * dQ.double()).view(rows_q, Hkv, G * D).sum(2))
    sum_dV = torch.zeros_like(sum_dO)
    sum_dK = torch.zeros_like(sum_dO)
    abs_dK = torch.zeros_like(sum_dO)
    k_dk = torch.zeros_like(q_dq)
    for s in range(fr.n_steps):
        kseq = torch.from_numpy(np.ascontiguousarray(pl["steps"][s]["k_seq"]).astype(np.int64)).cuda()
        sum_dV.index_add_(0, kseq, dVs[s].double())
        sum_dK.index_add_(0, kseq, dKs[s].double())
        abs_dK.index_add_(0, kseq, dKs[s].double().abs())
        k_dk.index_add_(0, kseq, (fr.Kd[s].double() * dKs[s].double()).sum(2))
    e_dv = float((sum_dV - sum_dO).norm() / sum_dO.norm())
    e_dk = float(sum_dK.abs().sum() / abs_dK.sum())
    e_qk = float((q_dq - k_dk).norm() / q_dq.norm())
    print(f"cfg{cfg}: identities over every key row: sum dV {e_dv:.1e}, sum dK {e_dk:.1e}, "
          f"Q.dQ=K.dK {e_qk:.1e}")
    # bf16 rounding of every dK/dV/dQ element (2^-9 relative, zero mean) is all that separates
    # the two sides of an identity
    assert e_dv <= 2e-3, f"cfg{cfg}: sum dV identity off by {e_dv}"
    assert e_dk <= 2e-3, f"cfg{cfg}: sum dK identity off by {e_dk}"
    assert e_qk <= 1e-2, f"cfg{cfg}: Q.dQ = K.dK identity off by {e_qk}"


def _check_sparse_dO(fr, n_random, n_boundary, groups=None):
    """dO non-zero on a sampled row set R only; every dK / dV element of every
    ring step, and dQ of R, against the oracle evaluated on the rows of R over all keys."""
    U, cfg, Hq, Hkv, D, rows_q = fr.U, fr.cfg, fr.Hq, fr.Hkv, fr.D, fr.rows_q
    G = Hq // Hkv
    R = _sample_rows(fr.pl, n_random, fr.w.seed + 7, n_boundary)
    ridx = torch.from_numpy(R).cuda()
    dO_sp = torch.zeros_like(fr.dO)
    dO_sp[ridx] = fr.dO[ridx]
    dQ, dKs, dVs = fr.backward(dO_sp, clear_in_prep=True)
    # dQ of rows outside R: dS = P (dP - delta) = 0 exactly
    mask = torch.ones(rows_q, dtype=torch.bool, device="cuda")
    mask[ridx] = False
    assert float(dQ[mask].float().abs().max()) == 0.0, "dQ outside the rows with dO != 0 is not 0"
    ks, kp = fr.key_meta()
    kblk = fr.key_blocks()
    qs, qp = fr.opl["q_seq"][R], fr.opl["q_pos"][R]
    Q3, dO3 = fr.Qb.reshape(rows_q, Hq, D)[R], fr.dOb.reshape(rows_q, Hq, D)[R]
    got_dQ = fr.bits_of(dQ[ridx]).reshape(len(R), Hq, D)
    # the oracle's formulas under the LSE and delta = rowsum(dO o O) the kernel was given for the
    # rows of R (gpu_util.grad_compare says why); O and LSE themselves are checked on sampled rows
    lse_R = fr.LSE[:, ridx].double().cpu().numpy()
    dl_R = (fr.bits_of(fr.O[ridx]).reshape(len(R), Hq, D) * oracle.bf16_to_f64(dO3)).sum(-1).T
    for g in (range(Hkv) if groups is None else groups):
        hs = slice(g * G, (g + 1) * G)
        Kg, Vg = fr.kv_heads(fr.Kb, [g]), fr.kv_heads(fr.Vb, [g])
        dQo, dKo, dVo = oracle.attn_bwd(np.ascontiguousarray(Q3[:, hs]), Kg, Vg,
                                        np.ascontiguousarray(dO3[:, hs]), qs, qp, ks, kp,
                                        LSE=np.ascontiguousarray(lse_R[hs]),
                                        delta=np.ascontiguousarray(dl_R[hs]))
        label = f"cfg{cfg} sparse dO ({len(R)} rows), KV head {g}: "
        U.grad_compare("dQ", got_dQ[:, hs], dQo, np.arange(len(R)), label)
        gk = np.concatenate([fr.bits_of(d[:, g]).reshape(-1, 1, D) for d in dKs])
        U.grad_compare("dK", gk, dKo, kblk, label)
        gv = np.concatenate([fr.bits_of(d[:, g]).reshape(-1, 1, D) for d in dVs])
        U.grad_compare("dV", gv, dVo, kblk, label)
        del Kg, Vg, dKo, dVo, gk, gv


def test_cfg2_full_size():
    fr = FullRun(2)
    fr.forward()
    dQ, dKs, dVs = fr.backward(fr.dO, clear_in_prep=False)
    _check_sampled_rows(fr, dQ, 24, 24)
    _check_identities(fr, dQ, dKs, dVs)
    # four whole heads, every element (SURVEY section 4 tier T2)
    U, D, rows = fr.U, fr.D, fr.rows_q
    heads = [0, 11, 22, 31]
    qs, qp = fr.opl["q_seq"], fr.opl["q_pos"]
    pick = lambda bits: np.ascontiguousarray(bits.reshape(rows, fr.Hq, D)[:, heads])  # noqa: E731
    Qh, dOh, Kh, Vh = pick(fr.Qb), pick(fr.dOb), pick(fr.Kb[0]), pick(fr.Vb[0])
    hidx = torch.tensor(heads, device="cuda")
    label = f"cfg2 heads {heads}, all {rows} rows: "
    got_O = fr.bits_of(fr.O[:, hidx]).reshape(rows, len(heads), D)
    got_L = fr.LSE[hidx].double().cpu().numpy()
    Oo, Lo = oracle.attn_fwd(Qh, Kh, Vh, qs, qp, qs, qp)
    U.o_compare(got_O, Oo, label)
    err_L = float(np.abs(got_L - Lo).max())
    assert err_L <= U.TOL_LSE, f"cfg2: LSE abs err {err_L}"
    print(f"{label}LSE abs err {err_L:.1e}")
    blk = U._blocks(0, qs, len(fr.w.seqs))
    got = [fr.bits_of(t[:, hidx]).reshape(rows, len(heads), D) for t in (dQ, dKs[0], dVs[0])]
    dl = np.ascontiguousarray((got_O * oracle.bf16_to_f64(dOh)).sum(-1).T)
    for strict, ref in ((False, oracle.attn_bwd(Qh, Kh, Vh, dOh, qs, qp, qs, qp)),
                        (True, oracle.attn_bwd(Qh, Kh, Vh, dOh, qs, qp, qs, qp, LSE=got_L, delta=dl))):
        for name, g, want in zip(("dQ", "dK", "dV"), got, ref):
            U.grad_compare(name, g, want, blk, label, strict)


def test_cfg3_full_size():
    fr = FullRun(3)
    fr.forward()
    dQ, dKs, dVs = fr.backward(fr.dO, clear_in_prep=False)
    _check_sampled_rows(fr, dQ, 6, 24)
    _check_identities(fr, dQ, dKs, dVs)
    del dQ, dKs, dVs
    _check_sparse_dO(fr, 24, 8)


def test_cfg4_full_size():
    fr = FullRun(4)
    fr.forward()
    dQ, dKs, dVs = fr.backward(fr.dO, clear_in_prep=False)
    _check_sampled_rows(fr, dQ, 6, 24)
    _check_identities(fr, dQ, dKs, dVs)


def test_cfg5_full_size():
    fr = FullRun(5)
    fr.forward()
    dQ, dKs, dVs = fr.backward(fr.dO, clear_in_prep=False)
    _check_sampled_rows(fr, dQ, 1, 3)  # ~1e11 fp64 flop of oracle per sampled row at 2M keys
    _check_identities(fr, dQ, dKs, dVs)
    del dQ, dKs, dVs
    # two of the eight KV groups (the oracle pass over 2M keys costs ~25 s per group; the other
    # groups' dK / dV are covered by the identities above and, element-wise, by the twins)
    _check_sparse_dO(fr, 8, 6, groups=(0, 5))
