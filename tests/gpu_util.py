"""Helpers of the -m gpu parity tests: build a workload's tensors once (seeded generator), run
the CUDA path through the C-ABI binding, run the oracle on the same inputs, compare."""
import numpy as np
import torch

import oracle
from paper_2502_21231_b200 import binding as B
from paper_2502_21231_b200.synth import rng, workloads

# BASELINE.json north_star tolerances
TOL_O = 1.5e-2      # max abs
TOL_LSE = 1e-3      # abs
TOL_GRAD = 1e-2     # relative L2


def to_dev(bits):
    """uint16 bf16 bit patterns (numpy) -> torch.bfloat16 CUDA tensor."""
    return torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16)


def to_bits(t):
    return t.detach().view(torch.int16).cpu().numpy().view(np.uint16)


def bf16_round(x):
    """fp64 -> nearest bf16 (ties to even) -> fp64; used to report the output-format floor."""
    b = np.asarray(x, np.float32).view(np.uint32).astype(np.uint64)
    b = (b + 0x7FFF + ((b >> 16) & 1)) & 0xFFFF0000
    return b.astype(np.uint32).view(np.float32).astype(np.float64)


def rel_l2(got, want):
    want = np.asarray(want, np.float64)
    got = np.asarray(got, np.float64)
    den = np.sqrt((want ** 2).sum())
    return float(np.sqrt(((got - want) ** 2).sum()) / den) if den > 0 else float(np.abs(got).max())


class DeviceRun:
    """One simulated rank: local Q/dO, per-step K/V, plan from the LIBRARY (bs_plan)."""

    def __init__(self, w, steps=None, gen_kv=True, fused_clear=False):
        self.w = w
        self.fused_clear = fused_clear  # dQ_acc cleared by the first bs_attn_fwd instead of prep
        self.dQ_acc = None
        self.plan = B.plan(w.seqs)
        self.Hq, self.Hkv, self.D = w.n_q_heads, w.n_kv_heads, w.head_dim
        pl = self.plan
        self.q_rows = pl["q_rows"]
        qruns = workloads.runs_from(pl["q_seq"], pl["q_pos"])
        self.Q_bits = workloads.gen_rows(w.seed, rng.STREAM_Q, qruns, self.Hq * self.D)
        self.dO_bits = workloads.gen_rows(w.seed, rng.STREAM_DO, qruns, self.Hq * self.D)
        self.steps = list(range(pl["n_steps"])) if steps is None else steps
        self.K_bits, self.V_bits = {}, {}
        if gen_kv:
            for s in self.steps:
                st = pl["steps"][s]
                kruns = workloads.runs_from(st["k_seq"], st["k_pos"])
                self.K_bits[s] = workloads.gen_rows(w.seed, rng.STREAM_K, kruns, self.Hkv * self.D)
                self.V_bits[s] = workloads.gen_rows(w.seed, rng.STREAM_V, kruns, self.Hkv * self.D)

    def shape(self, step):
        return B.make_shape(self.Hq, self.Hkv, self.D, self.q_rows,
                            self.plan["steps"][step]["kv_rows"])

    def q3(self, bits):
        return bits.reshape(-1, self.Hq, self.D)

    def kv3(self, bits):
        return bits.reshape(-1, self.Hkv, self.D)

    def forward(self, merge=True):
        """Run every step's bs_attn_fwd and (if more than one step) bs_lse_merge.
        Returns (O bf16 cuda [q_rows,Hq,D], LSE f32 cuda [Hq,q_rows], per-step partials)."""
        Q = to_dev(self.Q_bits)
        parts = []
        if self.fused_clear:
            self.dQ_acc = torch.full((self.q_rows, self.Hq, self.D), float("nan"),
                                     dtype=torch.float32, device="cuda")
        for s in self.steps:
            st = self.plan["steps"][s]
            sh = self.shape(s)
            K, V = to_dev(self.K_bits[s]), to_dev(self.V_bits[s])
            O = torch.full((self.q_rows, self.Hq, self.D), float("nan"), dtype=torch.bfloat16,
                           device="cuda")
            LSE = torch.full((self.Hq, self.q_rows), float("nan"), dtype=torch.float32,
                             device="cuda")
            ws = torch.empty(B.attn_workspace_bytes(sh, len(st["segs"]), False), dtype=torch.uint8,
                             device="cuda")
            B.attn_fwd(sh, Q, K, V, st["segs"], (0, self.q_rows), O, LSE, ws,
                       self.dQ_acc if (self.fused_clear and s == self.steps[0]) else None)
            parts.append((O, LSE))
        torch.cuda.synchronize()
        if len(parts) == 1 or not merge:
            return parts[0][0], parts[0][1], parts
        O = torch.empty_like(parts[0][0])
        LSE = torch.empty_like(parts[0][1])
        B.lse_merge([p[0] for p in parts], [p[1] for p in parts], self.shape(self.steps[0]),
                    (0, self.q_rows), O, LSE)
        torch.cuda.synchronize()
        return O, LSE, parts

    def backward(self, O, LSE):
        """prep, every step's bs_attn_bwd, finish.  Returns dQ bf16, {step: (dK, dV)}."""
        Q, dO = to_dev(self.Q_bits), to_dev(self.dO_bits)
        sh0 = self.shape(self.steps[0])
        delta = torch.empty((self.Hq, self.q_rows), dtype=torch.float32, device="cuda")
        if self.fused_clear:
            dQ_acc = self.dQ_acc
            B.attn_bwd_prep(sh0, O, dO, delta, None)
        else:
            dQ_acc = torch.full((self.q_rows, self.Hq, self.D), float("nan"), dtype=torch.float32,
                                device="cuda")
            B.attn_bwd_prep(sh0, O, dO, delta, dQ_acc)
        grads = {}
        for s in self.steps:
            st = self.plan["steps"][s]
            sh = self.shape(s)
            K, V = to_dev(self.K_bits[s]), to_dev(self.V_bits[s])
            dK = torch.full_like(K.view(-1, self.Hkv, self.D), float("nan"))
            dV = torch.full_like(dK, float("nan"))
            ws = torch.empty(B.attn_workspace_bytes(sh, len(st["segs"]), True), dtype=torch.uint8,
                             device="cuda")
            B.attn_bwd(sh, Q, K, V, dO, LSE, delta, st["segs"], dQ_acc, dK, dV, ws)
            grads[s] = (dK, dV)
        dQ = torch.empty((self.q_rows, self.Hq, self.D), dtype=torch.bfloat16, device="cuda")
        B.attn_bwd_finish(sh0, dQ_acc, dQ)
        torch.cuda.synchronize()
        return dQ, grads, delta

    # ------------------------------------------------------------------ oracle side
    def oracle_all_keys(self):
        """(K_bits, V_bits, k_seq, k_pos) of the union of all steps' KV buffers, taken from the
        ORACLE planner (independent of the library's plan)."""
        opl = oracle.oracle_plan(self.w.seqs)
        ks = np.concatenate([opl["steps"][s]["k_seq"] for s in self.steps])
        kp = np.concatenate([opl["steps"][s]["k_pos"] for s in self.steps])
        Kb = np.concatenate([self.K_bits[s] for s in self.steps])
        Vb = np.concatenate([self.V_bits[s] for s in self.steps])
        return opl, Kb, Vb, ks, kp

    def oracle_forward(self, rows=None):
        opl, Kb, Vb, ks, kp = self.oracle_all_keys()
        qs, qp = opl["q_seq"], opl["q_pos"]
        Qb = self.q3(self.Q_bits)
        if rows is not None:
            qs, qp, Qb = qs[rows], qp[rows], Qb[rows]
        return oracle.attn_fwd(Qb, self.kv3(Kb), self.kv3(Vb), qs, qp, ks, kp)

    def oracle_backward(self, LSE=None, delta=None):
        """Plain definition over all keys (LSE = delta = None), or the same formulas under a given
        normaliser LSE and a given delta ([Hq, q_rows] fp64): what a6 computes from ITS inputs."""
        opl, Kb, Vb, ks, kp = self.oracle_all_keys()
        dQ, dK, dV = oracle.attn_bwd(self.q3(self.Q_bits), self.kv3(Kb), self.kv3(Vb),
                                     self.q3(self.dO_bits), opl["q_seq"], opl["q_pos"], ks, kp,
                                     LSE=LSE, delta=delta)
        # split dK/dV back per step
        out, row = {}, 0
        for s in self.steps:
            n = opl["steps"][s]["kv_rows"]
            out[s] = (dK[row:row + n], dV[row:row + n])
            row += n
        return dQ, out


def o_compare(got_O, Oo, label=""):
    """O against the oracle, element by element.  BASELINE.json's bound is 1.5e-2 max-abs.  A bf16
    output cannot meet it where the output FORMAT alone is off by more: half an ulp is 1.5625e-2
    for |O| in [4, 8).  DESIGN.md reading 19: the strict bound holds for every element except
    those whose own quantisation floor |bf16(O_oracle) - O_oracle| exceeds 1.5e-2 - 4e-3; those
    are bounded by their floor + 4e-3.  Prints how many elements that concerns, the largest error
    among the strictly bounded ones and the floor, and asserts.  Returns the max abs error."""
    diff = np.abs(got_O - Oo)
    floor = np.abs(bf16_round(Oo) - Oo)
    loose = floor > TOL_O - 4e-3
    tol = np.where(loose, floor + 4e-3, TOL_O)
    n_big = int((np.abs(Oo) >= 4.0).sum())
    strict_max = float(diff[~loose].max()) if (~loose).any() else 0.0
    print(f"{label}O: {diff.size} elements, max abs err {float(diff.max()):.3e} (strict bound "
          f"{TOL_O}: max {strict_max:.3e} over {int((~loose).sum())} elements); |O| >= 4: {n_big} "
          f"elements; bf16 quantisation floor of the oracle values: max {float(floor.max()):.3e}, "
          f"{int(loose.sum())} elements above {TOL_O - 4e-3:.1e} (bounded by floor + 4e-3)")
    assert np.all(diff <= tol), (f"{label}O max abs err {float(diff.max())}; worst excess over the "
                                 f"per-element bound {float((diff - tol).max())}")
    return float(diff.max())


def grad_compare(name, got, want, block_of_row, label="", strict=True):
    """One gradient tensor [rows, heads, D] against an oracle tensor: relative L2 over the whole
    tensor (BASELINE.json: <= 1e-2) and - strict - over every block x head (block_of_row: e.g.
    (ring step, document, 128-row chunk), so that a broken short document cannot hide behind a
    long one), plus an element-wise bound.  A block whose oracle gradient is identically zero (a
    length-1 document's dQ / dK) must be zero to 1e-4 rms.  Element-wise: P, dS and the result are
    each rounded to bf16 (half an ulp: up to 2^-8 relative), so an element that one term dominates
    may be off by 3 x 2^-8 of its value, and an element that many terms make up by a random walk
    of such steps over terms whose root-sum-square is of the order of the block's rms:
    |err| <= 3 x 2^-8 |want| + 0.08 rms(block).
    strict=False (comparison with the PLAIN definition): only the whole-tensor bound is asserted
    and the worst block is printed.  Why: delta = rowsum(dO o O) is formed from the bf16 output O
    (as flash-attention backward does, and as a5 is defined), and dS = P (dP - delta) cancels when
    one key dominates a row, so a two-token document's gradient can be smaller than the error
    2^-9 |dO||O| that O's output rounding alone puts into delta.  The strict per-block and
    element-wise bounds are therefore asserted against the oracle's formulas evaluated under the
    LSE and delta the backward kernel was actually given (check_backward)."""
    got = np.asarray(got, np.float64)
    want = np.asarray(want, np.float64)
    assert got.shape == want.shape and got.ndim == 3
    assert not np.isnan(got).any(), f"{label}{name} has NaN"
    whole = rel_l2(got, want)
    blk = np.asarray(block_of_row, np.int64)
    nb = int(blk.max()) + 1 if len(blk) else 0
    H, D = got.shape[1], got.shape[2]
    num = np.zeros((nb, H))
    den = np.zeros((nb, H))
    cnt = np.bincount(blk, minlength=nb).astype(np.float64)[:, None] * D
    np.add.at(num, blk, ((got - want) ** 2).sum(-1))
    np.add.at(den, blk, (want ** 2).sum(-1))
    live = cnt[:, 0] > 0
    zero = (den == 0) & live[:, None]
    rel = np.sqrt(num / np.where(den > 0, den, 1.0))
    rel[~(den > 0)] = 0.0
    worst = float(rel.max()) if rel.size else 0.0
    zero_rms = float(np.sqrt((num / np.maximum(cnt, 1))[zero]).max()) if zero.any() else 0.0
    rms = np.sqrt(den / np.maximum(cnt, 1))                     # [blocks, heads]
    # (absolute floor: fp32 cancellation noise where the oracle gradient is exactly zero, e.g. the
    # first row of a document, whose dS = P (dP - delta) is 0 only in exact arithmetic)
    bound = 3 * 2.0 ** -8 * np.abs(want) + 0.08 * rms[blk][:, :, None] + 1e-5
    ratio = float((np.abs(got - want) / bound).max()) if got.size else 0.0
    kind = "given LSE/delta" if strict else "plain definition"
    print(f"{label}{name} vs {kind}: rel-L2 whole {whole:.2e}, worst block x head {worst:.2e} over "
          f"{int(live.sum())} x {H}, zero-gradient blocks rms {zero_rms:.1e}, "
          f"element-wise err / bound max {ratio:.2f}")
    assert whole <= TOL_GRAD, f"{label}{name} relative L2 error {whole} ({kind})"
    if strict:
        assert worst <= TOL_GRAD, (f"{label}{name} relative L2 error {worst} in block x head "
                                   f"{np.unravel_index(int(rel.argmax()), rel.shape)}")
        assert zero_rms <= 1e-4, f"{label}{name}: block with zero oracle gradient has rms {zero_rms}"
        assert ratio <= 1.0, f"{label}{name}: element-wise error {ratio} x the bound"
    return whole


def host_delta(O, dO_bits, rows, Hq, D):
    """delta[h, i] = sum_d dO[i,h,d] * O[i,h,d] in fp64 from the bf16 O the device returned."""
    o = oracle.bf16_to_f64(to_bits(O)).reshape(rows, Hq, D)
    do = oracle.bf16_to_f64(dO_bits).reshape(rows, Hq, D)
    return np.ascontiguousarray((o * do).sum(-1).T)


def check_forward(run, O, LSE, rows=None, label=""):
    Oo, Lo = run.oracle_forward(rows)
    got_O = oracle.bf16_to_f64(to_bits(O)).reshape(run.q_rows, run.Hq, run.D)
    got_L = LSE.double().cpu().numpy()
    if rows is not None:
        got_O, got_L = got_O[rows], got_L[:, rows]
    assert not np.isnan(got_O).any() and not np.isnan(got_L).any()
    err_O = o_compare(got_O, Oo, label)
    fin = np.isfinite(Lo)
    assert np.array_equal(np.isneginf(got_L), np.isneginf(Lo))
    err_L = float(np.abs(got_L[fin] - Lo[fin]).max()) if fin.any() else 0.0
    assert np.all(got_O[~fin.T] == 0)
    assert err_L <= TOL_LSE, f"{label}LSE abs err {err_L}"
    return err_O, err_L


def _blocks(step_idx, seq, n_seq):
    """Block id per row: (step, document, 128-row chunk of the document's rows in the buffer)."""
    seq = np.asarray(seq, np.int64)
    n = len(seq)
    start = np.zeros(n, np.int64)  # index of the first row of each run of equal seq
    if n:
        brk = np.flatnonzero(seq[1:] != seq[:-1]) + 1
        first = np.concatenate(([0], brk))
        start = np.repeat(first, np.diff(np.concatenate((first, [n]))))
    chunk = (np.arange(n) - start) // 128
    key = (step_idx * n_seq + seq) * (n // 128 + 2) + chunk
    _, ids = np.unique(key, return_inverse=True)
    return ids


def check_backward(run, dQ, grads, O, LSE, label=""):
    """dQ, dK, dV of a DeviceRun against the oracle over all keys.
    (i) the plain definition: whole-tensor relative L2 (BASELINE.json's tolerance);
    (ii) the same formulas under the LSE and delta = rowsum(dO o O) that bs_attn_bwd was given
    (O, LSE: the forward's merged outputs, themselves checked by check_forward): whole tensor,
    every (ring step, document, 128-row chunk) x head block, and element by element.
    Returns the whole-tensor errors of (i)."""
    opl = oracle.oracle_plan(run.w.seqs)
    n_seq = len(run.w.seqs)
    qblk = _blocks(0, opl["q_seq"], n_seq)
    kblk, base = [], 0
    for s in run.steps:
        b = _blocks(0, opl["steps"][s]["k_seq"], n_seq) + base
        base = int(b.max()) + 1 if len(b) else base
        kblk.append(b)
    kblk = np.concatenate(kblk)
    got_dQ = oracle.bf16_to_f64(to_bits(dQ)).reshape(run.q_rows, run.Hq, run.D)
    got = {}
    for i, n in ((0, "dK"), (1, "dV")):
        got[n] = np.concatenate([oracle.bf16_to_f64(to_bits(grads[s][i])).reshape(-1, run.Hkv, run.D)
                                 for s in run.steps])
    errs = {}
    lse64 = LSE.double().cpu().numpy()
    dl64 = host_delta(O, run.dO_bits, run.q_rows, run.Hq, run.D)
    for strict, (dQo, go) in ((False, run.oracle_backward()),
                              (True, run.oracle_backward(LSE=lse64, delta=dl64))):
        e = {"dQ": grad_compare("dQ", got_dQ, dQo, qblk, label, strict)}
        for i, n in ((0, "dK"), (1, "dV")):
            e[n] = grad_compare(n, got[n], np.concatenate([go[s][i] for s in run.steps]), kblk,
                                label, strict)
        if not strict:
            errs = e
    return errs
