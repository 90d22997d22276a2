#!/usr/bin/env python
"""bench.py — one JSON line for the driver.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Workload: BASELINE.json configs[1] (the 7B-shaped packed batch the metric is quoted on):
32768-token buffer, log-normal document lengths, 32/32 heads, head_dim 128, bf16, fwd + bwd.
A "step" is one pass of the whole hot path: bs_plan (host) -> bs_attn_fwd -> bs_attn_bwd_prep ->
bs_attn_bwd -> bs_attn_bwd_finish (cfg2 has one ring step, so the LSE merge is not on its path;
the merge is timed separately on the cfg3-shaped partials and reported under "merge").
value = unmasked FLOPs (14 * D * Hq * visible pairs) of all ranks / max-over-ranks device time.
N > 1: every rank runs its own cfg2-shaped batch (weak scaling, no data-path collective —
HDP ranks are independent per micro-batch); torch.distributed is used only for
the barrier and the max-over-ranks of the device time.
--impl reference: times the fp64 oracle (the reference arm of this tier) on the host cores.
--gpus N with N > 1 and no WORLD_SIZE in the environment: bench.py starts the N ranks itself
(python -m torch.distributed.run, one process per GPU, rendezvous on 127.0.0.1).
--impl plumbing: the launch path alone on CPU (gloo): every rank times a host-only step (bs_plan),
barrier, max over ranks, rank 0 prints the line - what tests/test_dist_gloo.py drives with 2 ranks.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "varlen causal attn fwd+bwd TFLOP/s (unmasked)"
WORKLOAD = "cfg2_7B_packed_32k"
ORACLE_SAMPLE_HEADS = 1  # heads of cfg2 per step of the reference arm (MHA heads are independent)
CPU_BASELINE_HEADS = 5    # heads the cpu_baseline leg of the default run times (~12 s)
# bs_assign replay: global batch, rank capacity and number of HDP ranks
HDP_CAPACITY, HDP_RANKS, HDP_N_SHORT, HDP_LONG_MULTIPLES = 8192, 16, 384, (8, 4, 2, 2)


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(tflops=d["bf16_tflops"], tflops_sustained=d.get("bf16_tflops_sustained"),
                    hbm=d["hbm_gbs"], source="measured (MEASURED_PEAKS.json)")
    return dict(tflops=1590.0, tflops_sustained=1400.0, hbm=6650.0,
                source="fallback (B200_PROFILING.md)")


def ncu_traffic(kernel_prefix):
    """DRAM bytes (read + write) per launch of a kernel from this round's ncu capture
    (profiles/r02_traffic.csv: kernel, dram__bytes_read.sum, dram__bytes_write.sum, sha256[:16] of
    the kernel's source file at capture time), or None.  It cannot be measured inside this run
    (no profiler here); a capture of OTHER source than the one that is running is not reported."""
    import hashlib
    path = os.path.join(ROOT, "profiles", "r02_traffic.csv")
    try:
        for line in open(path).read().splitlines()[1:]:
            f = line.split(",")
            if f[0].startswith(kernel_prefix):
                src = os.path.join(ROOT, "paper_2502_21231_b200", "csrc", f[3])
                if hashlib.sha256(open(src, "rb").read()).hexdigest()[:16] != f[4].strip():
                    return None
                return int(f[1]) + int(f[2])
    except (OSError, ValueError, IndexError):
        pass
    return None


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag = index, [], set(), False
        self.stamps, self.max_mhz = [], None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                     nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                     nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                     nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap"}
            while not self.stop_flag:
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                self.stamps.append(time.perf_counter())
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
                time.sleep(0.02)
        except Exception as e:  # NVML missing: report nothing rather than fail the bench
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")

    def median_between(self, t0, t1):
        s = sorted(v for v, t in zip(self.samples, self.stamps) if t0 <= t <= t1)
        return s[len(s) // 2] if s else None

    def result(self):
        s = sorted(self.samples)
        return dict(sm_mhz=s[len(s) // 2] if s else None, sm_max_mhz=self.max_mhz,
                    reasons=sorted(self.reasons))


def cfg2():
    from paper_2502_21231_b200.synth import make_workload
    return make_workload(2)


def oracle_sample_run(w, heads, want_time=True):
    """Oracle fwd + bwd on the first `heads` heads of cfg2 (all 32768 tokens).  Returns
    (seconds, flops, threads)."""
    import numpy as np
    import oracle
    from paper_2502_21231_b200.synth import rng, workloads
    pl = oracle.oracle_plan(w.seqs)
    D = w.head_dim
    runs = workloads.runs_from(pl["q_seq"], pl["q_pos"])
    full = w.n_q_heads * D

    def gen(stream):
        return workloads.gen_rows(w.seed, stream, runs, full).reshape(-1, w.n_q_heads, D)[:, :heads].copy()
    Q, K, V, dO = gen(rng.STREAM_Q), gen(rng.STREAM_K), gen(rng.STREAM_V), gen(rng.STREAM_DO)
    t0 = time.perf_counter()
    oracle.attn_fwd(Q, K, V, pl["q_seq"], pl["q_pos"], pl["q_seq"], pl["q_pos"])
    oracle.attn_bwd(Q, K, V, dO, pl["q_seq"], pl["q_pos"], pl["q_seq"], pl["q_pos"])
    dt = time.perf_counter() - t0
    pairs = pl["steps"][0]["visible_pairs"]
    return dt, 14.0 * D * heads * pairs, oracle.threads()


def run_reference(args, rank):
    if rank != 0:
        return
    w = cfg2()
    times = []
    for i in range(args.warmup + args.steps):
        dt, flops, thr = oracle_sample_run(w, ORACLE_SAMPLE_HEADS)
        if i >= args.warmup:
            times.append(dt)
    t = sum(times) / len(times)
    val = flops / t / 1e12
    sample = (f"{ORACLE_SAMPLE_HEADS} of {w.n_q_heads} heads of {WORKLOAD}, all 32768 tokens, "
              "fwd+bwd, fp64")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": "TFLOP/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": val, "unit": "TFLOP/s", "cores": thr, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": val, "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_ours(args, rank, world, local_rank):
    import numpy as np
    import torch
    from paper_2502_21231_b200 import binding as B
    from paper_2502_21231_b200 import dist_util as DU
    from paper_2502_21231_b200.synth import rng, workloads

    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    w = cfg2()
    Hq, Hkv, D = w.n_q_heads, w.n_kv_heads, w.head_dim
    seed = DU.rank_seed(w.seed, rank)  # same document lengths on every rank, different tensors
    pl = B.plan(w.seqs)
    st = pl["steps"][0]
    rows, pairs = pl["q_rows"], st["visible_pairs"]
    qruns = workloads.runs_from(pl["q_seq"], pl["q_pos"])

    def host(stream, heads):
        bits = workloads.gen_rows(seed, stream, qruns, heads * D)
        return torch.from_numpy(bits.view(np.int16)).view(torch.bfloat16).view(rows, heads, D).pin_memory()
    hQ, hK, hV, hdO = host(rng.STREAM_Q, Hq), host(rng.STREAM_K, Hkv), host(rng.STREAM_V, Hkv), host(rng.STREAM_DO, Hq)
    Q, K, V, dO = (t.cuda() for t in (hQ, hK, hV, hdO))
    O, dQ = torch.empty_like(Q), torch.empty_like(Q)
    dK, dV = torch.empty_like(K), torch.empty_like(K)
    LSE = torch.empty((Hq, rows), dtype=torch.float32, device="cuda")
    delta = torch.empty_like(LSE)
    acc = torch.empty((rows, Hq, D), dtype=torch.float32, device="cuda")
    sh = B.make_shape(Hq, Hkv, D, rows, rows)
    ws_f = torch.empty(B.attn_workspace_bytes(sh, len(st["segs"]), False), dtype=torch.uint8, device="cuda")
    ws_b = torch.empty(B.attn_workspace_bytes(sh, len(st["segs"]), True), dtype=torch.uint8, device="cuda")
    hO, hdQ, hdK, hdV = (torch.empty_like(t, device="cpu").pin_memory() for t in (O, dQ, dK, dV))
    ev = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731

    def step(marks=None):
        p = B.plan(w.seqs)["steps"][0]["segs"]  # a1: host planning is part of the step
        if marks:
            marks[0].record()
        B.attn_fwd(sh, Q, K, V, p, (0, rows), O, LSE, ws_f, acc)  # also clears the dQ accumulator
        if marks:
            marks[1].record()
        B.attn_bwd_prep(sh, O, dO, delta, None)
        if marks:
            marks[2].record()
        B.attn_bwd(sh, Q, K, V, dO, LSE, delta, p, acc, dK, dV, ws_b)
        if marks:
            marks[3].record()
        B.attn_bwd_finish(sh, acc, dQ)
        if marks:
            marks[4].record()

    def barrier():
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    marks = [[ev() for _ in range(5)] for _ in range(args.steps)]
    B.launch_count_reset()
    e0, e1 = ev(), ev()
    e0.record()
    for i in range(args.steps):
        step(marks[i])
    e1.record()
    barrier()
    launches = B.launch_count()
    ms = e0.elapsed_time(e1)
    t_fwd = sum(m[0].elapsed_time(m[1]) for m in marks) / args.steps
    t_prep = sum(m[1].elapsed_time(m[2]) for m in marks) / args.steps
    t_bwd = sum(m[2].elapsed_time(m[3]) for m in marks) / args.steps
    t_fin = sum(m[3].elapsed_time(m[4]) for m in marks) / args.steps
    if args.only_step:
        sampler.stop_flag = True
        sampler.join()
        (ms,) = DU.max_over_ranks(dist, [ms], "cuda")
        if rank == 0:
            fl = 14.0 * D * Hq * pairs
            print(json.dumps({"metric": METRIC, "value": world * fl * args.steps / (ms * 1e-3) / 1e12,
                              "unit": "TFLOP/s", "n_gpus": world, "steps": args.steps,
                              "ms_per_step": ms / args.steps, "only_step": True,
                              "kernels_ms": {"bs_attn_fwd": t_fwd, "bs_attn_bwd_prep": t_prep,
                                             "bs_attn_bwd": t_bwd, "bs_attn_bwd_finish": t_fin},
                              "gpu_launches": launches, "clocks": sampler.result()}))
        if dist:
            dist.barrier()
            dist.destroy_process_group()
        return
    # sustained leg (north_star: "sustains"): the same step back to back for >= 2 s, so that the
    # part sits at its power cap; reported against the measured SUSTAINED bf16 peak
    n_sus = max(args.steps, int(2200.0 / (ms / args.steps)))
    s0, s1 = ev(), ev()
    t_sus0 = time.perf_counter()
    s0.record()
    for _ in range(n_sus):
        step()
    s1.record()
    barrier()
    t_sus1 = time.perf_counter()
    ms_sus = s0.elapsed_time(s1)
    # end to end: every step copies its inputs from pinned host memory, runs, and copies its results
    # back, all inside the timed region.  The copies are PCIe-bound (1 GiB each way per step), so the
    # steps are software-pipelined over three streams with two sets of device buffers: while step i
    # computes, step i+1's inputs come in and step i-1's results go out.
    s_in, s_run, s_out = (torch.cuda.Stream() for _ in range(3))
    sets = []
    for _ in range(2):
        d = dict(Q=torch.empty_like(Q), K=torch.empty_like(K), V=torch.empty_like(V), dO=torch.empty_like(dO),
                 O=torch.empty_like(O), dQ=torch.empty_like(dQ), dK=torch.empty_like(dK), dV=torch.empty_like(dV),
                 LSE=torch.empty_like(LSE), delta=torch.empty_like(delta), acc=torch.empty_like(acc),
                 ws_f=torch.empty_like(ws_f), ws_b=torch.empty_like(ws_b),
                 in_ready=torch.cuda.Event(), ran=torch.cuda.Event(), out_done=torch.cuda.Event())
        sets.append(d)

    def e2e_step(i):
        d = sets[i & 1]
        with torch.cuda.stream(s_in):
            s_in.wait_event(d["ran"])           # step i-2 no longer reads these inputs
            for k, h in (("Q", hQ), ("K", hK), ("V", hV), ("dO", hdO)):
                d[k].copy_(h, non_blocking=True)
            d["in_ready"].record(s_in)
        with torch.cuda.stream(s_run):
            s_run.wait_event(d["in_ready"])
            s_run.wait_event(d["out_done"])     # step i-2's results have left the output buffers
            p = B.plan(w.seqs)["steps"][0]["segs"]
            B.attn_fwd(sh, d["Q"], d["K"], d["V"], p, (0, rows), d["O"], d["LSE"], d["ws_f"], d["acc"])
            B.attn_bwd_prep(sh, d["O"], d["dO"], d["delta"], None)
            B.attn_bwd(sh, d["Q"], d["K"], d["V"], d["dO"], d["LSE"], d["delta"], p, d["acc"], d["dK"],
                       d["dV"], d["ws_b"])
            B.attn_bwd_finish(sh, d["acc"], d["dQ"])
            d["ran"].record(s_run)
        with torch.cuda.stream(s_out):
            s_out.wait_event(d["ran"])
            for h, k in ((hO, "O"), (hdQ, "dQ"), (hdK, "dK"), (hdV, "dV")):
                h.copy_(d[k], non_blocking=True)
            d["out_done"].record(s_out)

    for i in range(2):
        e2e_step(i)
    barrier()
    f0, f1 = ev(), ev()
    f0.record()
    for s_ in (s_in, s_run, s_out):
        s_.wait_event(f0)
    for i in range(args.steps):
        e2e_step(i)
    cur = torch.cuda.current_stream()
    for s_ in (s_in, s_run, s_out):
        e_ = torch.cuda.Event()
        e_.record(s_)
        cur.wait_event(e_)
    f1.record()
    barrier()
    ms_e2e = f0.elapsed_time(f1)
    sampler.stop_flag = True
    sampler.join()
    ms, ms_e2e, ms_sus = DU.max_over_ranks(dist, [ms, ms_e2e, ms_sus], "cuda")
    flops_step = 14.0 * D * Hq * pairs
    out = None
    if rank == 0:
        pk = peaks()
        nb = lambda t: t.numel() * t.element_size()  # noqa: E731
        merge = bench_merge(B, torch, pk)
        red_dram = bench_reduce_probe(B, torch, acc)            # 512 MiB: every line misses L2
        red_l2 = bench_reduce_probe(B, torch, acc[:4096])       # 64 MiB: the accumulator stays in L2
        xent = bench_softmax_xent(B, torch, pk)
        ring = bench_ring_steps(B, torch, workloads, pk)
        full = bench_full_configs(B, torch, workloads, pk)
        # naive HDP assignment (bs_assign) of a synthetic global batch,
        # every rank's micro-batches replayed on this GPU
        from paper_2502_21231_b200 import replay as RP
        hdp_lens = RP.global_batch(w.seed, HDP_N_SHORT, HDP_CAPACITY, HDP_LONG_MULTIPLES)
        hdp = RP.replay(hdp_lens, HDP_CAPACITY, HDP_RANKS, Hq, Hkv, D, seed=w.seed)
        hdp_bal = RP.replay_balanced(hdp_lens, HDP_CAPACITY, HDP_RANKS, Hq, Hkv, D, seed=w.seed)
        # the static-CP packed baseline on the same global batch, and whether
        # the O(S^2) compute hides the O(S) PCIe copies of an activation offload
        static_cp = RP.static_cp_baseline(hdp_lens, HDP_CAPACITY, HDP_RANKS, HDP_RANKS, Hq, Hkv, D,
                                          seed=w.seed)
        offload = RP.offload_probe((8192, 32768, 65536), Hq, Hkv, D, seed=w.seed)
        hdp["workload"] = (f"{HDP_N_SHORT} log-normal short sequences + long ones of "
                           f"{list(HDP_LONG_MULTIPLES)} x capacity, capacity {HDP_CAPACITY} tokens, "
                           f"d_hdp {HDP_RANKS}, {Hq} heads, D {D}")
        dt, fl, thr = oracle_sample_run(w, CPU_BASELINE_HEADS)
        bwd_tflops = 10.0 * D * Hq * pairs / (t_bwd * 1e-3) / 1e12
        fwd_tflops = 4.0 * D * Hq * pairs / (t_fwd * 1e-3) / 1e12
        value = world * flops_step * args.steps / (ms * 1e-3) / 1e12
        sus = world * flops_step * n_sus / (ms_sus * 1e-3) / 1e12
        prep_bytes = rows * Hq * (4 * D + 4)          # reads O, dO; writes delta (dQ_acc cleared by fwd)
        bwd_red_bytes = tile_area_ratio(w) * pairs / (128 * 128) * Hq * 128 * D * 4   # tile-blocks x 64 KB
        fin_bytes = rows * Hq * 6 * D                 # reads fp32 dQ_acc, writes bf16 dQ
        # The driver keeps the contract keys of this line and the END of stdout: the long replay
        # records come first, what explains the headline (kernels, sustained, merge) sits inside
        # "roofline" and at the end.
        out = {
            "metric": METRIC, "value": value,
            "unit": "TFLOP/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {"workload": WORKLOAD, "tokens": rows, "documents": len(w.seqs),
                       "n_q_heads": Hq, "n_kv_heads": Hkv, "head_dim": D,
                       "visible_pairs_per_head": pairs, "flops_per_step": flops_step,
                       "computed_over_visible": tile_area_ratio(w),
                       "l2": "inputs+outputs 2.4 GB per step exceed the 126 MB L2; no flush",
                       "peaks": pk["source"]},
            "full_configs": full,
            "ring_steps_cfg3_4_5": ring,
            "hdp_naive_replay": hdp,
            "hdp_balance_replay": hdp_bal,
            "static_cp_baseline": static_cp,
            "offload_probe": offload,
            "softmax_xent": xent,
            "merge": merge,
            "pct_of_bf16_peak": {"measured_burst": 100 * value / world / pk["tflops"],
                                 "nominal_2250": 100 * value / world / 2250.0},
            "roofline": {"kernel": "attn_bwd_kernel<128>", "bound": "tensor", "achieved": bwd_tflops,
                         "peak": pk["tflops"], "unit": "TFLOP/s", "frac": bwd_tflops / pk["tflops"],
                         "traffic": ncu_traffic("attn_bwd_kernel"),
                         "kernels": {
                             "bs_attn_fwd": {"ms": round(t_fwd, 4), "tflops": round(fwd_tflops, 1),
                                             "frac": round(fwd_tflops / pk["tflops"], 4)},
                             "bs_attn_bwd_prep": {"ms": round(t_prep, 4),
                                                  "gbs": round(prep_bytes / t_prep / 1e6, 1)},
                             "bs_attn_bwd": {"ms": round(t_bwd, 4), "tflops": round(bwd_tflops, 1),
                                             "frac": round(bwd_tflops / pk["tflops"], 4)},
                             "bs_attn_bwd_finish": {"ms": round(t_fin, 4),
                                                    "gbs": round(fin_bytes / t_fin / 1e6, 1)}},
                         "sustained": {"tflops": round(sus, 1), "seconds": round(ms_sus * 1e-3, 2),
                                       "steps": n_sus,
                                       "frac_of_sustained_peak": round(sus / world / pk["tflops_sustained"], 4)
                                       if pk["tflops_sustained"] else None,
                                       "frac_of_burst_peak": round(sus / world / pk["tflops"], 4),
                                       "sm_mhz_median": sampler.median_between(t_sus0, t_sus1)},
                         # the backward's other ceiling: every computed 128 x 128
                         # tile-block adds 128 x D fp32 of partial dQ into dQ_acc in the L2 atomic
                         # units; the probes are that traffic alone (bs_reduce_probe), one CTA per SM,
                         # units, L2-resident (64 MiB) and not (the whole 512 MiB accumulator)
                         "l2_reduce": {"bytes_per_launch": int(bwd_red_bytes),
                                       "achieved_gbs": round(bwd_red_bytes / t_bwd / 1e6, 1),
                                       "probe_all_miss_gbs": round(red_dram, 1),
                                       "probe_l2_resident_gbs": round(red_l2, 1),
                                       "frac_of_all_miss_probe": round(bwd_red_bytes / t_bwd / 1e6 / red_dram, 4),
                                       "frac_of_l2_resident_probe": round(bwd_red_bytes / t_bwd / 1e6 / red_l2, 4)},
                         "merge_gbs": {k: {"gbs": v["gbs"], "of_n_to_1_probe": v["frac_of_n_to_1_probe"],
                                               "of_measured_copy": v["frac_of_measured_copy"]}
                                           for k, v in merge["by_config"].items()}},
            "cpu_baseline": {"value": fl / dt / 1e12, "unit": "TFLOP/s", "cores": thr, "kind": "oracle",
                             "sample": f"{CPU_BASELINE_HEADS} of {Hq} heads of {WORKLOAD}, all "
                                       f"{rows} tokens, fwd+bwd, fp64, {dt:.1f} s"},
            "e2e": {"value": world * flops_step * args.steps / (ms_e2e * 1e-3) / 1e12, "unit": "TFLOP/s",
                    "h2d_bytes_per_step": sum(nb(t) for t in (Q, K, V, dO)),
                    "d2h_bytes_per_step": sum(nb(t) for t in (O, dQ, dK, dV))},
            "gpu_launches": launches, "clocks": sampler.result()}
    if dist:
        dist.barrier()
        dist.destroy_process_group()
    if out:
        print(json.dumps(out))


def bench_merge(B, torch, pk):
    """bs_lse_merge on the partials of configs 3, 4, 5 (n = 8 / 4 / 64 parts; rows x heads 32768 x 64,
    65536 x 32, 32768 x 48; D = 128), each next to two plain streaming probes with the same byte
    counts and the merge's own load instruction (bs_hbm_probe): n input streams read
    and one written (n : 1), and n + 1 streams only read.  The probes say what a read-dominated
    kernel can reach on this part; the merge is reported against them and against the measured
    copy bandwidth."""
    ev = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731

    def timed(fn, it=10):
        for _ in range(3):
            fn()
        a, b = ev(), ev()
        a.record()
        for _ in range(it):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / it

    out, D = {}, 128
    sink = torch.zeros(4, dtype=torch.uint8, device="cuda")
    for cfg, n, rows, Hq in ((3, 8, 32768, 64), (4, 4, 65536, 32), (5, 64, 32768, 48)):
        Os = [torch.randn((rows, Hq, D), device="cuda").to(torch.bfloat16) for _ in range(n)]
        Ls = [torch.randn((Hq, rows), device="cuda") for _ in range(n)]
        O, L = torch.empty_like(Os[0]), torch.empty_like(Ls[0])
        sh = B.make_shape(Hq, 8, D, rows, rows)
        ms = timed(lambda: B.lse_merge(Os, Ls, sh, (0, rows), O, L), 10 if n < 64 else 4)
        ms_alias = timed(lambda: B.lse_merge(Os, Ls, sh, (0, rows), Os[0], Ls[0]), 10 if n < 64 else 4)
        nbytes = (n + 1) * rows * Hq * (2 * D + 4)
        ms_n1 = timed(lambda: B.hbm_probe(Os, O, sink), 10 if n < 64 else 4)
        rd = (Os + [O])[:B.BS_MAX_MERGE_PARTS]          # n + 1 streams, at most 64
        ms_rd = timed(lambda: B.hbm_probe(rd, None, sink), 10 if n < 64 else 4)
        pbytes = (n + 1) * rows * Hq * 2 * D
        rbytes = len(rd) * rows * Hq * 2 * D
        gbs = nbytes / ms / 1e6
        out[f"cfg{cfg}"] = {"n_parts": n, "rows": rows, "heads": Hq, "ms": round(ms, 4), "bytes": nbytes,
                            "gbs": round(gbs, 1), "gbs_output_aliases_part0": round(nbytes / ms_alias / 1e6, 1),
                            "probe_n_to_1_gbs": round(pbytes / ms_n1 / 1e6, 1),
                            "probe_pure_read_gbs": round(rbytes / ms_rd / 1e6, 1),
                            "frac_of_n_to_1_probe": round(gbs / (pbytes / ms_n1 / 1e6), 4),
                            "frac_of_measured_copy": round(gbs / pk["hbm"], 4),
                            "frac_of_nominal_8000": round(gbs / 8000.0, 4)}
        del Os, Ls, O, L
        torch.cuda.empty_cache()
    c3 = out["cfg3"]
    return {"workload": "partials of cfg3 / cfg4 / cfg5, D = 128; probes = bs_hbm_probe, same bytes",
            "by_config": out,
            "roofline": {"bound": "hbm", "achieved": c3["gbs"], "peak": pk["hbm"], "unit": "GB/s",
                         "frac": c3["gbs"] / pk["hbm"], "frac_of_nominal_8000": c3["gbs"] / 8000.0,
                         "traffic": ncu_traffic("lse_merge_kernel")}}


def bench_reduce_probe(B, torch, acc):
    """bs_reduce_probe: GB/s of fp32 reduce-adds (TMA boxes of 16 KB into `acc`, one CTA per SM, the
    backward's own instruction and box shape) with nothing else running."""
    boxes = 256
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    for _ in range(3):
        B.reduce_probe(acc, boxes)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    it = 10
    a.record()
    for _ in range(it):
        B.reduce_probe(acc, boxes)
    b.record()
    b.synchronize()
    return n_sm * boxes * 16384 * it / (a.elapsed_time(b) * 1e-3) / 1e9


def tile_area_ratio(w):
    """Pairs the attention kernels COMPUTE on this workload / pairs that are visible (and counted):
    masked halves of diagonal tiles and ragged document tails earn nothing ("FLOPs
    proportional to the areas of attention mask").  Both kernels visit every (128-row query tile,
    128-key block) pair of a document with at least one visible element, whole.  Whole documents
    (cp = 1) only."""
    computed = vis = 0
    for L, cp, _ in w.seqs:
        assert cp == 1
        n = -(-L // 128)
        vis += L * (L + 1) // 2
        computed += 128 * 128 * (n * (n + 1) // 2)
    return round(computed / vis, 4)


def bench_softmax_xent(B, torch, pk):
    """bs_softmax_xent: 32768 tokens x 16384 logits (a 128K
    vocabulary under TP = 8), bf16 in / bf16 gradients out, 2.1 GB per call (> L2)."""
    T, V = 32768, 16384
    x = (torch.randn(T, V, device="cuda") * 3).bfloat16()
    y = torch.randint(0, V, (T,), device="cuda", dtype=torch.int32)
    loss, d = torch.empty(T, device="cuda"), torch.empty_like(x)
    for _ in range(3):
        B.softmax_xent(x, y, 1.0 / T, loss, d)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    it = 10
    e0.record()
    for _ in range(it):
        B.softmax_xent(x, y, 1.0 / T, loss, d)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / it
    nbytes = T * V * 4 + T * 8
    gbs = nbytes / (ms * 1e-3) / 1e9
    del x, d
    torch.cuda.empty_cache()
    return {"workload": f"{T} tokens x {V} logits (128K vocabulary / TP 8), bf16", "ms": ms,
            "bytes": nbytes,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm"], "unit": "GB/s",
                         "frac": gbs / pk["hbm"], "frac_of_nominal_8000": gbs / 8000.0,
                         "traffic": ncu_traffic("softmax_xent")}}


def bench_full_configs(B, torch, workloads, pk, cfgs=(1, 3, 4, 5)):
    """every config as a WHOLE pipeline on seeded-shape random device data - all ring
    steps of bs_attn_fwd (the first one clears dQ_acc), bs_lse_merge over all partials, prep, all
    ring steps of bs_attn_bwd, finish - each phase timed once with CUDA events after one untimed
    warm-up pass of the same launches.  cfg1 is forward only and latency-bound: microseconds."""
    out = {}
    ev = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731
    for cfg in cfgs:
        w = workloads.make_workload(cfg)
        pl = B.plan(w.seqs)
        Hq, Hkv, D, rows, n = w.n_q_heads, w.n_kv_heads, w.head_dim, pl["q_rows"], pl["n_steps"]
        Q = torch.randn(rows, Hq, D, device="cuda").bfloat16()
        dO = torch.randn_like(Q)
        acc = torch.empty((rows, Hq, D), dtype=torch.float32, device="cuda")
        steps = []
        for st in pl["steps"]:
            K = torch.randn(st["kv_rows"], Hkv, D, device="cuda").bfloat16()
            sh = B.make_shape(Hq, Hkv, D, rows, st["kv_rows"])
            nb = max(B.attn_workspace_bytes(sh, len(st["segs"]), False),
                     B.attn_workspace_bytes(sh, len(st["segs"]), True))
            steps.append(dict(st=st, sh=sh, K=K, V=torch.randn_like(K), dK=torch.empty_like(K),
                              dV=torch.empty_like(K), O=torch.empty_like(Q),
                              L=torch.empty((Hq, rows), dtype=torch.float32, device="cuda"),
                              ws=torch.empty(nb, dtype=torch.uint8, device="cuda")))
        sh0 = steps[0]["sh"]
        # merged rows: the rows that take part in more than one step (cfg4: the long shard only)
        m_end = max(sg[1] for d in steps[1:] for sg in d["st"]["segs"]) if n > 1 else 0
        # running merge: the output aliases part 0 (include/bytescale_attn.h), so rows that are
        # final after step 0 (cfg4's short documents) need no copy
        O, LSE = steps[0]["O"], steps[0]["L"]
        delta = torch.empty_like(LSE)
        dQ = torch.empty_like(Q)

        def fwd():
            for i, d in enumerate(steps):
                B.attn_fwd(d["sh"], Q, d["K"], d["V"], d["st"]["segs"], (0, rows if i == 0 else m_end),
                           d["O"], d["L"], d["ws"], acc if i == 0 else None)

        def merge():
            if n > 1:
                B.lse_merge([d["O"] for d in steps], [d["L"] for d in steps], sh0, (0, m_end), O, LSE)

        def bwd():
            B.attn_bwd_prep(sh0, O, dO, delta, None)
            for d in steps:
                B.attn_bwd(d["sh"], Q, d["K"], d["V"], dO, LSE, delta, d["st"]["segs"], acc, d["dK"],
                           d["dV"], d["ws"])
            B.attn_bwd_finish(sh0, acc, dQ)

        phases = (fwd,) if cfg == 1 else (fwd, merge, bwd)
        reps = 20 if cfg == 1 else 1
        for f in phases:  # warm-up pass
            f()
        torch.cuda.synchronize()
        t = []
        for f in phases:
            a, b = ev(), ev()
            a.record()
            for _ in range(reps):
                f()
            b.record()
            torch.cuda.synchronize()
            t.append(a.elapsed_time(b) / reps)
        pairs = sum(st["visible_pairs"] for st in pl["steps"])
        if cfg == 1:
            out["cfg1"] = {"fwd_us": round(1e3 * t[0], 2), "visible_pairs_per_head": pairs,
                           "note": "latency-bound correctness config: 960 tokens, 4 heads, D 64"}
            continue
        mbytes = (n + 1) * m_end * Hq * (2 * D + 4)
        both = 14.0 * D * Hq * pairs / (t[0] + t[2]) / 1e9
        out[f"cfg{cfg}"] = {
            "ring_steps": n, "visible_pairs_per_head": pairs,
            "fwd_ms": round(t[0], 3), "merge_ms": round(t[1], 3), "bwd_ms": round(t[2], 3),
            "fwd_tflops": round(4.0 * D * Hq * pairs / t[0] / 1e9, 1),
            "bwd_tflops": round(10.0 * D * Hq * pairs / t[2] / 1e9, 1),
            "fwd_bwd_tflops": round(both, 1), "frac_of_measured_peak": round(both / pk["tflops"], 3),
            "merge_gbs": round(mbytes / t[1] / 1e6, 1), "merge_bytes": mbytes}
        del steps, Q, dO, acc, O, LSE, delta, dQ
        torch.cuda.empty_cache()
    return out


def bench_ring_steps(B, torch, workloads, pk):
    """Configs 3-5 (GQA long sequences, zigzag CP): one diagonal (step 0) and one off-diagonal
    (step 1) ring step each, bs_attn_fwd and bs_attn_bwd timed with CUDA events on seeded-shape
    random device data.  Context for the headline number (which is cfg2): unmasked TFLOP/s."""
    out = {}
    ev = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731

    def timed(fn, n=3):
        fn()
        torch.cuda.synchronize()
        a, b = ev(), ev()
        a.record()
        for _ in range(n):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / n

    for cfg in (3, 4, 5):
        w = workloads.make_workload(cfg)
        pl = B.plan(w.seqs)
        Hq, Hkv, D, rows = w.n_q_heads, w.n_kv_heads, w.head_dim, pl["q_rows"]
        Q = torch.randn(rows, Hq, D, device="cuda").bfloat16()
        dO = torch.randn_like(Q)
        O = torch.empty_like(Q)
        LSE = torch.full((Hq, rows), 8.0, dtype=torch.float32, device="cuda")
        delta = torch.zeros_like(LSE)
        acc = torch.zeros((rows, Hq, D), dtype=torch.float32, device="cuda")
        for sidx in (0, 1):
            st = pl["steps"][sidx]
            kv, segs, pairs = st["kv_rows"], st["segs"], st["visible_pairs"]
            K = torch.randn(kv, Hkv, D, device="cuda").bfloat16()
            V = torch.randn_like(K)
            dK, dV = torch.empty_like(K), torch.empty_like(K)
            sh = B.make_shape(Hq, Hkv, D, rows, kv)
            wsf = torch.empty(B.attn_workspace_bytes(sh, len(segs), False), dtype=torch.uint8, device="cuda")
            wsb = torch.empty(B.attn_workspace_bytes(sh, len(segs), True), dtype=torch.uint8, device="cuda")
            tf = timed(lambda: B.attn_fwd(sh, Q, K, V, segs, (0, rows), O, LSE, wsf))
            tb = timed(lambda: B.attn_bwd(sh, Q, K, V, dO, LSE, delta, segs, acc, dK, dV, wsb))
            f_tf, b_tf = 4.0 * D * Hq * pairs / tf / 1e9, 10.0 * D * Hq * pairs / tb / 1e9
            both = 14.0 * D * Hq * pairs / (tf + tb) / 1e9
            out[f"cfg{cfg}_step{sidx}"] = {"fwd_ms": round(tf, 3), "bwd_ms": round(tb, 3),
                                          "fwd_tflops": round(f_tf, 1), "bwd_tflops": round(b_tf, 1),
                                          "fwd_bwd_tflops": round(both, 1),
                                          "frac_of_measured_peak": round(both / pk["tflops"], 3)}
        del Q, dO, O, LSE, delta, acc
        torch.cuda.empty_cache()
    return out


def run_plumbing(args, rank, world):
    """The multi-rank launch path alone, on CPU (gloo): what --gpus N does around the timed region
    - rendezvous, barrier, max over ranks, one line from rank 0 - with a host-only step (bs_plan
    of cfg2) in place of the device work.  tests/test_dist_gloo.py drives it with 2 ranks."""
    import torch.distributed as dist
    from paper_2502_21231_b200 import binding as B
    from paper_2502_21231_b200 import dist_util as DU
    if world > 1:
        dist.init_process_group("gloo")
    else:
        dist = None
    w = cfg2()
    for _ in range(max(args.warmup, 1)):
        B.plan(w.seqs)
    if dist:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        pl = B.plan(w.seqs)
    ms = (time.perf_counter() - t0) * 1e3
    (ms_max,) = DU.max_over_ranks(dist, [ms], "cpu")
    if dist:
        dist.barrier()
    if rank == 0:
        print(json.dumps({"impl": "plumbing", "metric": "bs_plan calls/s (host only)",
                          "value": DU.whole_job_rate(args.steps, world, ms_max), "unit": "calls/s",
                          "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 1),
                          "ms_per_step": ms_max / args.steps, "higher_is_better": True,
                          "scaling": "weak", "q_rows": pl["q_rows"], "gpu_launches": 0}))
    if dist:
        dist.destroy_process_group()


def launch_ranks(args):
    """--gpus N > 1 without a launcher: start N ranks of this script under torch.distributed.run
    (one process per GPU, rendezvous on 127.0.0.1) and pass their output through."""
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
           f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1", "--master-port", str(port),
           os.path.abspath(__file__), "--gpus", str(args.gpus), "--steps", str(args.steps),
           "--warmup", str(args.warmup), "--impl", args.impl] + (["--only-step"] if args.only_step else [])
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference", "plumbing"])
    ap.add_argument("--only-step", action="store_true",
                    help="time the cfg2 step only (no sustained / e2e / merge / replay / oracle legs): "
                         "the short command the ncu captures under profiles/ are taken with")
    args = ap.parse_args()
    if args.impl != "reference" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(launch_ranks(args))
    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    local_rank = int(os.environ.get("LOCAL_RANK", 0))
    if args.impl == "reference":
        run_reference(args, rank)
    elif args.impl == "plumbing":
        run_plumbing(args, rank, world)
    else:
        if world > 1:
            # NCCL only carries the barrier and the max over ranks; its communicator log stays on
            # so that the number of ranks that really joined can be read from the run's output
            os.environ.setdefault("NCCL_DEBUG", "INFO")
            os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
