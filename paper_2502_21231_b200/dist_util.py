"""Multi-rank plumbing of bench.py (replicas only: HDP ranks are independent per micro-batch,
PAPER.md:161-165; the ring exchange of KV chunks is outside this build's scope).  Nothing here
touches the data path: a barrier, the max-over-ranks of the device times, per-rank seeds."""
import torch


def rank_seed(base_seed: int, rank: int) -> int:
    """Same document lengths on every rank (the length stream is drawn from base_seed by the
    workload), different tensor contents."""
    return base_seed + 100 * rank


def max_over_ranks(dist, values, device):
    """Element-wise max of a list of floats over all ranks (dist may be None: single process)."""
    if dist is None:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def whole_job_rate(units_per_rank: float, world: int, ms_max: float) -> float:
    """Weak scaling: every rank processes units_per_rank in the slowest rank's time."""
    return world * units_per_rank / (ms_max * 1e-3)
