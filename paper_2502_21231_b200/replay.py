"""Replay of a `bs_assign` result on one GPU: every micro-batch of every HDP rank is planned
(`bs_plan`) and run through the attention hot path (forward of every ring step + LSE merge, then
prep / backward of every ring step / finish), one after the other, timed with CUDA events.  The
per-rank totals give the picture of PAPER.md:405 (naive HDP: "significant time variance across
ranks ... min=60s, max=279s, std=68s") for this library's kernels on a synthetic global batch.

What is replayed is each rank's own compute; the ring exchange of K/V chunks between ranks is
outside the north_star, so the K/V buffer of a step holds seeded random rows of the right count.
Timing only: parity of the sharded path against the oracle is the job of tests/."""
import math

import torch

from . import binding as B


def global_batch(seed, n_short, capacity, long_multiples):
    """Synthetic global batch (stand-in for the long-tailed length histograms of PAPER.md:85,107,
    which are not available here): `n_short` log-normal lengths clipped to [64, capacity], and one
    sequence of m * capacity tokens for every m in `long_multiples`; input order shuffled."""
    g = torch.Generator().manual_seed(seed)
    mu, sigma = math.log(capacity / 8.0), 1.0
    short = torch.exp(mu + sigma * torch.randn(n_short, generator=g)).clamp(64, capacity).long()
    lens = [int(x) for x in short] + [int(m * capacity) for m in long_multiples]
    perm = torch.randperm(len(lens), generator=g)
    return [lens[int(i)] for i in perm]


def _prepare_step(seqs, Hq, Hkv, D, gen, out):
    """Buffers and the step closure of one micro-batch: out[0] = step, returns visible pairs."""
    pl = B.plan([(s[0], s[1], s[2]) for s in seqs])
    rows, n_steps = pl["q_rows"], pl["n_steps"]
    if rows == 0:
        out[0] = None
        return 0
    dev = "cuda"
    Q = torch.randn(rows, Hq, D, device=dev, generator=gen).bfloat16()
    dO = torch.randn(rows, Hq, D, device=dev, generator=gen).bfloat16()
    Ks, Vs, shapes, ws_f, ws_b = [], [], [], [], []
    for st in pl["steps"]:
        kv = st["kv_rows"]
        Ks.append(torch.randn(kv, Hkv, D, device=dev, generator=gen).bfloat16())
        Vs.append(torch.randn(kv, Hkv, D, device=dev, generator=gen).bfloat16())
        sh = B.make_shape(Hq, Hkv, D, rows, kv)
        shapes.append(sh)
        ws_f.append(torch.empty(B.attn_workspace_bytes(sh, len(st["segs"]), False), dtype=torch.uint8,
                                device=dev))
        ws_b.append(torch.empty(B.attn_workspace_bytes(sh, len(st["segs"]), True), dtype=torch.uint8,
                                device=dev))
    parts_O = [torch.empty_like(Q) for _ in range(n_steps)]
    parts_L = [torch.empty((Hq, rows), dtype=torch.float32, device=dev) for _ in range(n_steps)]
    O = torch.empty_like(Q) if n_steps > 1 else parts_O[0]
    LSE = torch.empty_like(parts_L[0]) if n_steps > 1 else parts_L[0]
    delta = torch.empty_like(parts_L[0])
    acc = torch.empty((rows, Hq, D), dtype=torch.float32, device=dev)
    dQ = torch.empty_like(Q)
    dKs, dVs = [torch.empty_like(k) for k in Ks], [torch.empty_like(v) for v in Vs]

    def step():
        for s, st in enumerate(pl["steps"]):
            B.attn_fwd(shapes[s], Q, Ks[s], Vs[s], st["segs"], (0, rows), parts_O[s], parts_L[s],
                       ws_f[s], acc if s == 0 else None)
        if n_steps > 1:
            B.lse_merge(parts_O, parts_L, shapes[0], (0, rows), O, LSE)
        B.attn_bwd_prep(shapes[0], O, dO, delta, None)
        for s, st in enumerate(pl["steps"]):
            B.attn_bwd(shapes[s], Q, Ks[s], Vs[s], dO, LSE, delta, st["segs"], acc, dKs[s], dVs[s],
                       ws_b[s])
        B.attn_bwd_finish(shapes[0], acc, dQ)

    step()  # warm-up (first touch of the buffers)
    out[0] = step
    return sum(st["visible_pairs"] for st in pl["steps"])


def _run_microbatch(seqs, Hq, Hkv, D, gen):
    """One micro-batch on this GPU; returns (milliseconds, visible pairs per head)."""
    holder = [None]
    pairs = _prepare_step(seqs, Hq, Hkv, D, gen, holder)
    if holder[0] is None:
        return 0.0, 0
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    holder[0]()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b), pairs


def replay(lens, capacity, d_hdp, n_q_heads, n_kv_heads, head_dim, seed=0):
    """Runs every micro-batch of bs_assign(lens, capacity, d_hdp) and returns the per-rank picture:
    {"n_rounds", "rank_ms": [d_hdp], "min_ms", "max_ms", "mean_ms", "std_ms", "max_over_min",
     "idle_frac": share of rank-time spent waiting for the slowest rank, "tflops": unmasked
     fwd+bwd rate over the summed compute time}."""
    if not torch.cuda.is_available():
        raise RuntimeError("replay needs a CUDA device (there is no CPU path)")
    a = B.assign(lens, capacity, d_hdp)
    gen = torch.Generator(device="cuda").manual_seed(seed)
    rank_ms = [0.0] * d_hdp
    pairs = 0
    for rnd, rank, seqs in a["microbatches"]:
        ms, p = _run_microbatch(seqs, n_q_heads, n_kv_heads, head_dim, gen)
        rank_ms[rank] += ms
        pairs += p
    t = torch.tensor(rank_ms, dtype=torch.float64)
    busy = float(t.sum())
    return {"n_rounds": a["n_rounds"], "n_microbatches": len(a["microbatches"]),
            "ranks_needed_max": max(a["d"]) if a["d"] else 0,
            "rank_ms": [round(x, 3) for x in rank_ms],
            "min_ms": round(float(t.min()), 3), "max_ms": round(float(t.max()), 3),
            "mean_ms": round(float(t.mean()), 3), "std_ms": round(float(t.std(unbiased=False)), 3),
            "max_over_min": round(float(t.max() / t.min()), 2) if float(t.min()) > 0 else None,
            "idle_frac": round(1.0 - busy / (float(t.max()) * d_hdp), 3) if busy > 0 else None,
            "tflops": round(14.0 * head_dim * n_q_heads * pairs / (busy * 1e-3) / 1e12, 1)
            if busy > 0 else None}


def fit_cost_model(n_q_heads, n_kv_heads, head_dim, lengths=(512, 1024, 2048, 4096, 8192), seed=0):
    """T(s) = a2 s^2 + a1 s + a0 (Eq. 3) fitted by least squares to the measured
    fwd+bwd time of one whole sequence of s tokens on this GPU.  Returns non-negative integer
    coefficients in femtoseconds (the unit bs_balance schedules in) and the measured points."""
    gen = torch.Generator(device="cuda").manual_seed(seed)
    pts = []
    for s in lengths:
        ms = min(_run_microbatch([(s, 1, 0, 0)], n_q_heads, n_kv_heads, head_dim, gen)[0]
                 for _ in range(3))
        pts.append((s, ms))
    x = torch.tensor([[float(s) * s, float(s), 1.0] for s, _ in pts], dtype=torch.float64)
    y = torch.tensor([ms * 1e12 for _, ms in pts], dtype=torch.float64)   # ms -> fs
    coef = torch.linalg.lstsq(x, y.unsqueeze(1)).solution.squeeze(1)
    return [max(0, int(round(float(c)))) for c in coef], pts


def _timeline(microbatches, d_hdp, duration):
    """Per-rank finish times when the micro-batches run in schedule order and the ranks of a long
    sequence start together.  microbatches: [(rank, start, end, seqs)], duration(k) in ms."""
    order = sorted(range(len(microbatches)), key=lambda k: (microbatches[k][1], microbatches[k][0]))
    now = [0.0] * d_hdp
    busy = [0.0] * d_hdp
    gangs = {}
    for k in order:
        rank, _, _, seqs = microbatches[k]
        if seqs[0][1] > 1:
            gangs.setdefault(seqs[0][3], []).append(k)
    done = set()
    for k in order:
        if k in done:
            continue
        rank, _, _, seqs = microbatches[k]
        members = gangs[seqs[0][3]] if seqs[0][1] > 1 else [k]
        ranks = [microbatches[m][0] for m in members]
        start = max(now[r] for r in ranks)
        end = start + max(duration(m) for m in members)
        for m, r in zip(members, ranks):
            now[r] = end
            busy[r] += duration(m)
            done.add(m)
    return now, busy


def replay_balanced(lens, capacity, d_hdp, n_q_heads, n_kv_heads, head_dim, seed=0):
    """Algorithm 2 (bs_balance) on the cost model fitted to this GPU, next to Algorithm 1's own
    line 10 (bs_assign): makespans under the model, and the balanced schedule replayed on the GPU
    (every micro-batch run and timed, the ranks of a long sequence starting together)."""
    if not torch.cuda.is_available():
        raise RuntimeError("replay needs a CUDA device (there is no CPU path)")
    cost, pts = fit_cost_model(n_q_heads, n_kv_heads, head_dim, seed=seed)
    bal = B.balance(lens, capacity, d_hdp, cost)
    naive = B.assign(lens, capacity, d_hdp)

    def model_ms(seqs):
        t = sum(cost[0] * s[0] * s[0] + cost[1] * s[0] + cost[2] for s in seqs)
        return (t // seqs[0][1] if seqs[0][1] > 1 else t) * 1e-12
    naive_t = [0.0] * d_hdp
    for _, rank, seqs in naive["microbatches"]:
        naive_t[rank] += model_ms(seqs)
    gen = torch.Generator(device="cuda").manual_seed(seed)
    measured = [_run_microbatch(seqs, n_q_heads, n_kv_heads, head_dim, gen)[0]
                for _, _, _, seqs in bal["microbatches"]]
    finish, busy = _timeline(bal["microbatches"], d_hdp, lambda k: measured[k])
    t = torch.tensor(finish, dtype=torch.float64)
    return {"cost_fs": cost, "fit_points_ms": [(s, round(ms, 4)) for s, ms in pts],
            "model": {"naive_makespan_ms": round(max(naive_t), 3),
                      "balance_makespan_ms": round(bal["makespan"] * 1e-12, 3),
                      "speedup": round(max(naive_t) / (bal["makespan"] * 1e-12), 3)},
            "measured": {"rank_finish_ms": [round(x, 3) for x in finish],
                         "min_ms": round(float(t.min()), 3), "max_ms": round(float(t.max()), 3),
                         "std_ms": round(float(t.std(unbiased=False)), 3),
                         "max_over_min": round(float(t.max() / t.min()), 2) if float(t.min()) > 0 else None,
                         "idle_frac": round(1.0 - sum(busy) / (float(t.max()) * d_hdp), 3)},
            "n_microbatches": len(bal["microbatches"])}


def static_cp_baseline(lens, capacity, cp, d_hdp, n_q_heads, n_kv_heads, head_dim, seed=0):
    """The static parallelism HDP replaces (Fig. 14): the batch is packed into
    sequences of up to cp * capacity tokens, and EVERY document of a packed sequence is cut 2 cp
    ways over a CP group of cp ranks, however short it is.  Ranks of a group are symmetric
    (zigzag), so rank 0's micro-batch is run and timed for every packed sequence; the d_hdp / cp
    groups take the packed sequences round-robin.  Compute only: the ring exchange, which is
    what static CP wastes most on short documents, is outside this path."""
    if not torch.cuda.is_available():
        raise RuntimeError("replay needs a CUDA device (there is no CPU path)")
    packs, room = [[]], cp * capacity
    for s in sorted(lens, reverse=True):          # first-fit decreasing into cp * capacity tokens
        for pk in packs:
            if sum(pk) + s <= room:
                pk.append(s)
                break
        else:
            packs.append([s])
    packs = [pk for pk in packs if pk]
    gen = torch.Generator(device="cuda").manual_seed(seed)
    groups = max(1, d_hdp // cp)
    group_ms = [0.0] * groups
    pairs, rows = 0, 0
    for k, pk in enumerate(packs):
        ms, p = _run_microbatch([(s, cp, 0, i) for i, s in enumerate(pk)], n_q_heads, n_kv_heads,
                                head_dim, gen)
        group_ms[k % groups] += ms
        pairs += p
        rows += sum(pk) // cp
    busy = sum(group_ms)
    return {"cp": cp, "n_packed_sequences": len(packs), "groups": groups,
            "rank_ms": round(max(group_ms), 3),
            "tflops_per_rank": round(14.0 * head_dim * n_q_heads * pairs / (busy * 1e-3) / 1e12, 1)
            if busy > 0 else None}


def offload_probe(seq_lens, n_q_heads, n_kv_heads, head_dim, seed=0):
    """"the O(S^2) computation time will inevitably surpass the O(S) data transfer
    time".  For one whole sequence of S tokens: fwd+bwd compute time, the time to copy its Q, K, V
    and O (the activations an act_ctx would offload) to pinned host memory and back, and both at
    once on separate streams (the copies use the DMA engines)."""
    if not torch.cuda.is_available():
        raise RuntimeError("the probe needs a CUDA device")
    out = []
    gen = torch.Generator(device="cuda").manual_seed(seed)
    side = torch.cuda.Stream()
    for S in seq_lens:
        elems = S * (2 * n_q_heads + 2 * n_kv_heads) * head_dim      # Q, O, K, V
        dev = torch.empty(elems, dtype=torch.bfloat16, device="cuda")
        host = torch.empty(elems, dtype=torch.bfloat16, pin_memory=True)

        def copies():
            host.copy_(dev, non_blocking=True)       # D2H (forward: offload)
            dev.copy_(host, non_blocking=True)       # H2D (backward: reload)

        def timed(fn):
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b)
        compute_ms, _ = _run_microbatch([(S, 1, 0, 0)], n_q_heads, n_kv_heads, head_dim, gen)
        copies()
        copy_ms = timed(copies)

        def both():
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                copies()
            _run_once[0]()
            torch.cuda.current_stream().wait_stream(side)
        # one more micro-batch run whose step we can call again
        _run_once = [None]
        _prepare_step([(S, 1, 0, 0)], n_q_heads, n_kv_heads, head_dim, gen, _run_once)
        both_ms = timed(both)
        out.append({"tokens": S, "compute_ms": round(compute_ms, 3), "copy_ms": round(copy_ms, 3),
                    "both_ms": round(both_ms, 3), "bytes_each_way": elems * 2,
                    "overlap": round(max(compute_ms, copy_ms) / both_ms, 3),   # 1.0 = perfect
                    "copy_hidden_by_compute": compute_ms >= copy_ms})
        del dev, host
    return out
