"""CPU, world_size 2, gloo: the multi-rank plumbing bench.py uses for --gpus N (replicas only)."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    from paper_2502_21231_b200 import dist_util as DU
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, ms_e2e = 2.0 + rank, 10.0 - rank  # rank 1 is slower on-device, rank 0 end to end
    got = DU.max_over_ranks(dist, [ms, ms_e2e], "cpu")
    dist.barrier()
    seeds = [torch.tensor([DU.rank_seed(2504, rank)]) for _ in range(world)]
    dist.all_gather(seeds, torch.tensor([DU.rank_seed(2504, rank)]))
    if rank == 0:
        out.put((got, [int(s) for s in seeds], DU.whole_job_rate(1.75e12, world, got[0])))
    dist.destroy_process_group()


def test_max_over_ranks_and_seeds_world2():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got, seeds, rate = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got == [3.0, 10.0]           # max over ranks of each timing
    assert seeds == [2504, 2604]        # per-rank tensor seeds differ
    assert abs(rate - 2 * 1.75e12 / 3.0e-3) < 1.0   # whole-job rate uses the slowest rank's time


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    from paper_2502_21231_b200 import dist_util as DU
    assert DU.max_over_ranks(None, [1.5, 2], "cpu") == [1.5, 2.0]


def test_bench_gpus_2_starts_two_ranks():
    """`python bench.py --gpus 2` with no launcher around it starts the two ranks itself
    (torch.distributed.run on 127.0.0.1); here with --impl plumbing: the launch path, barrier and
    max-over-ranks of the real bench on CPU/gloo, a host-only step in place of the device work."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items()
           if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "3",
                        "--warmup", "1", "--impl", "plumbing"], capture_output=True, text=True,
                       timeout=300, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(x) for x in r.stdout.splitlines() if x.startswith("{")]
    assert len(lines) == 1, r.stdout          # rank 0 alone prints
    out = lines[0]
    assert out["n_gpus"] == 2 and out["steps"] == 3 and out["impl"] == "plumbing"
    assert out["value"] > 0 and out["q_rows"] == 32768
    # one process, no launcher, one GPU asked for: no spawn
    r1 = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "2", "--warmup", "1",
                         "--impl", "plumbing"], capture_output=True, text=True, timeout=300, env=env,
                        cwd=ROOT)
    assert r1.returncode == 0 and json.loads(r1.stdout.strip().splitlines()[-1])["n_gpus"] == 1
