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
