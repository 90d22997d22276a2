"""TEST INFRASTRUCTURE ONLY: plain Python restatement of the shard-descriptor rule (`bs_plan`).

Passages followed:
  * "Each subsequence of the packed sequences is uniformly divided into 2N parts and
    symmetrically assigned to the N devices.  It ensures that each device holds 1/N of all the
    subsequences and covers 1/N of the attention mask area.  All devices participate in the same
    ring-P2P communication, with the same data exchange volume."
  * CP "shards QKV along the sequence dimension ... KV slices ... exchanged across devices using
    a ring-style P2P communication"
  * HDP: short sequences stay whole on a rank next to slices of long ones
The paper gives no data structure; the canonical form is DESIGN.md "bs_plan canonical form"
(SURVEY.md 8(c).3): floor partition, low-then-high row order, source rank (r - s) mod N,
segments in (sequence, q part, k part) order, unclamped causal offset.

Pins (tests/test_plan.py): brute-force enumeration that the union over ranks and steps of the
visible (q_pos, k_pos) pairs is the causal set, each pair exactly once; the 1/N-tokens and
1/N-mask-area statements of PAPER.md:318; the worked examples in tests/golden/plan_examples.txt.
"""
import numpy as np


def parts_of(length, cp):
    """Global [begin,end) of every part of a sequence: 1 part if cp == 1, else 2*cp parts."""
    if cp == 1:
        return [(0, length)]
    return [((k * length) // (2 * cp), ((k + 1) * length) // (2 * cp)) for k in range(2 * cp)]


def held_parts(length, cp, p):
    """(low, high) global ranges held by rank p; high is empty (0,0) when cp == 1."""
    ps = parts_of(length, cp)
    if cp == 1:
        return ps[0], (0, 0)
    return ps[p], ps[2 * cp - 1 - p]


def _count_pairs(q_len, k_len, off):
    # per-row count, written out: row a sees keys b <= a + off, b in [0,k_len)
    total = 0
    for a in range(q_len):
        total += min(max(a + off + 1, 0), k_len)
    return total


def plan(seqs):
    """seqs: iterable of (len, cp, rank).  Returns a dict mirroring the C plan accessors."""
    seqs = [(int(a), int(b), int(c)) for a, b, c in seqs]
    for ln, cp, r in seqs:
        assert ln >= 1 and cp >= 1 and 0 <= r < cp
    cu_q = [0]
    q_seq, q_pos = [], []
    q_parts = []  # per seq: [(row_begin, global_begin, len) for low, high]
    for i, (ln, cp, r) in enumerate(seqs):
        row = cu_q[-1]
        entry = []
        for (b, e) in held_parts(ln, cp, r):
            entry.append((row, b, e - b))
            q_seq += [i] * (e - b)
            q_pos += list(range(b, e))
            row += e - b
        q_parts.append(entry)
        cu_q.append(row)
    n_steps = max([cp for _, cp, _ in seqs], default=0)
    steps = []
    for s in range(n_steps):
        segs, kv_seq, kv_src, cu_k, k_seq, k_pos = [], [], [], [0], [], []
        pairs = 0
        for i, (ln, cp, r) in enumerate(seqs):
            if cp <= s:
                continue
            p = (r - s) % cp
            kv_seq.append(i)
            kv_src.append(p)
            krow = cu_k[-1]
            k_parts = []
            for (b, e) in held_parts(ln, cp, p):
                k_parts.append((krow, b, e - b))
                k_seq += [i] * (e - b)
                k_pos += list(range(b, e))
                krow += e - b
            cu_k.append(krow)
            for (qrow, qg, ql) in q_parts[i]:
                for (kr, kg, kl) in k_parts:
                    if ql == 0 or kl == 0:
                        continue
                    if kg > qg + ql - 1:  # first key after the last query: nothing visible
                        continue
                    off = qg - kg
                    segs.append((qrow, qrow + ql, kr, kr + kl, off, i))
                    pairs += _count_pairs(ql, kl, off)
        steps.append(dict(step=s, segs=segs, kv_rows=cu_k[-1], kv_seq=kv_seq, kv_src_rank=kv_src,
                          cu_rows_k=cu_k, visible_pairs=pairs,
                          k_seq=np.asarray(k_seq, np.int32), k_pos=np.asarray(k_pos, np.int32)))
    return dict(n_seqs=len(seqs), q_rows=cu_q[-1], cu_rows_q=cu_q,
                q_seq=np.asarray(q_seq, np.int32), q_pos=np.asarray(q_pos, np.int32),
                n_steps=n_steps, steps=steps)
