"""Workload recipes: the five BASELINE.json configs (and scaled-down twins) as seeded synthetic
inputs.  Stand-ins for the paper's GitHub / Byted datasets, which are not
available; shapes follow Table 1 and the 256K-2048K contexts.

No arithmetic of the method lives here: a workload is a list of (len, cp, rank) sequences, head
counts and a seed; tensors are N(0,1) bf16 drawn per (sequence, global position) so any slice
can be generated on its own.  Which global rows a device holds is decided by the caller's plan
(the oracle's or the library's); `gen_rows` only fills the (seq, pos_begin, n_rows) runs it is
given.
"""
from dataclasses import dataclass, field
from typing import List, Tuple

import numpy as np

from . import rng


@dataclass
class Workload:
    name: str
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    seqs: List[Tuple[int, int, int]]  # (len, cp, rank)
    seed: int
    backward: bool = True
    note: str = ""
    extra: dict = field(default_factory=dict)


def runs_from(seq_arr, pos_arr):
    """Run-length encode per-row (seq, pos) arrays into [(seq, pos_begin, n_rows), ...]."""
    seq_arr = np.asarray(seq_arr)
    pos_arr = np.asarray(pos_arr)
    n = len(seq_arr)
    if n == 0:
        return []
    brk = np.flatnonzero((seq_arr[1:] != seq_arr[:-1]) | (pos_arr[1:] != pos_arr[:-1] + 1)) + 1
    starts = np.concatenate(([0], brk))
    ends = np.concatenate((brk, [n]))
    return [(int(seq_arr[s]), int(pos_arr[s]), int(e - s)) for s, e in zip(starts, ends)]


def gen_rows(seed, stream, runs, row_elems, out=None):
    """bf16 bits [sum n_rows, row_elems] for the given (seq, pos_begin, n_rows) runs."""
    total = sum(r[2] for r in runs)
    if out is None:
        out = np.empty((total, row_elems), np.uint16)
    assert out.shape == (total, row_elems)
    row = 0
    for seq, pos, n in runs:
        rng.rows_bf16(seed, stream, seq, pos, n, row_elems, out=out[row:row + n])
        row += n
    return out


def fill_lengths(draw, total, min_len):
    """Fill a buffer of exactly `total` tokens from an iterator of drawn lengths (DESIGN.md
    reading 7): take draws in order; truncate the last to the space left; if what is left is
    below min_len, add it to the previous document instead."""
    lens, used = [], 0
    for L in draw:
        L = int(L)
        left = total - used
        if L >= left:
            if left >= min_len or not lens:
                lens.append(left)
            else:
                lens[-1] += left
            return lens
        if left - L < min_len:  # the remainder could not form a document: absorb it now
            lens.append(left)
            return lens
        lens.append(L)
        used += L
    raise RuntimeError("length stream exhausted")


def lognormal_lengths(seed, total, median=1024.0, sigma=1.0, lo=128, hi=32768):
    z = rng.normal_f64(seed, rng.STREAM_LENGTHS, 0, 0, 4096)
    L = np.clip(np.rint(np.exp(np.log(median) + sigma * z)), lo, hi).astype(np.int64)
    return fill_lengths(iter(L), total, lo)


def pareto_lengths(seed, total, alpha=1.2, lo=64, hi=8192):
    u = rng.uniform_f64(seed, rng.STREAM_LENGTHS, 0, 0, 65536)
    L = np.minimum(np.floor(lo * u ** (-1.0 / alpha)), hi).astype(np.int64)
    return fill_lengths(iter(L), total, lo)


BASE_SEED = 2502


def make_workload(cfg: int) -> Workload:
    """BASELINE.json configs[cfg-1]."""
    if cfg == 1:
        return Workload("cfg1_tiny_packed_fwd", 4, 4, 64, [(64, 1, 0), (128, 1, 0), (256, 1, 0),
                                                            (512, 1, 0)], BASE_SEED + 1,
                        backward=False, note="4 documents {64,128,256,512}, MHA 4, D=64")
    if cfg == 2:
        lens = lognormal_lengths(BASE_SEED + 2, 32768)
        return Workload("cfg2_7B_packed_32k", 32, 32, 128, [(L, 1, 0) for L in lens],
                        BASE_SEED + 2, note="log-normal(median 1024, sigma 1.0) clip [128,32768]")
    if cfg == 3:
        return Workload("cfg3_gqa_cp8_256k", 64, 8, 128, [(262144, 8, 0)], BASE_SEED + 3,
                        note="one 262144-token sequence, CP=8, rank 0")
    if cfg == 4:
        lens = pareto_lengths(BASE_SEED + 4, 65536)
        return Workload("cfg4_hdp_mixed_128k", 32, 8, 128,
                        [(262144, 4, 1)] + [(L, 1, 0) for L in lens], BASE_SEED + 4,
                        note="65536-token CP=4 rank-1 shard + Pareto(1.2) documents in [64,8192]")
    if cfg == 5:
        return Workload("cfg5_2048k_cp64", 48, 8, 128, [(2097152, 64, 32)], BASE_SEED + 5,
                        note="one 2097152-token sequence, CP=64, rank 32")
    raise ValueError(cfg)


def scaled_twin(cfg: int, c: int = 256, ragged: bool = False, rank=None, kv_heads=None) -> Workload:
    """Same structure (N, r, Hq/Hkv ratio, D, segment pattern) as configs 3-5 with part length ~c.
    ragged=True makes 2N not divide L and c unaligned to any tile.  kv_heads: number of KV heads
    (the group size Hq/Hkv is kept; fewer groups make the fp64 oracle pass affordable)."""
    w = make_workload(cfg)
    ln, cp, r = w.seqs[0]
    assert cp > 1
    r = r if rank is None else rank
    L = 2 * cp * c + (cp + 3 if ragged else 0)
    if ragged:
        L -= 2 * cp * 7
    rest = []
    if cfg == 4:
        lens = pareto_lengths(w.seed + 100, 2 * c + (13 if ragged else 0), hi=max(64, c // 2))
        rest = [(x, 1, 0) for x in lens]
    group = w.n_q_heads // w.n_kv_heads
    hkv = w.n_kv_heads if kv_heads is None else kv_heads
    return Workload(f"{w.name}_twin_c{c}{'_ragged' if ragged else ''}_r{r}", hkv * group, hkv,
                    w.head_dim, [(L, cp, r)] + rest, w.seed + 1000 + r,
                    note=f"scaled twin of cfg{cfg}")


CONFIGS = (1, 2, 3, 4, 5)
