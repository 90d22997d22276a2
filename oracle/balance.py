"""TEST INFRASTRUCTURE ONLY: oracle of `bs_balance`, the balance strategy for HDP (PAPER.md
Algorithm 2, lines 290-304 of PAPER.md and section 6.3-6.4) in its DP-Balance form, which replaces
line 10 of Algorithm 1 ("instead of line 10 in Alg. 1").

Plain Python, integers only, in the order of the algorithm's lines.  What is scheduled are the
groups of Algorithm 1 lines 1-9 (oracle/assign.py: a long sequence on D(s) ranks, or a bin of
short ones on one rank).  Readings:

B1  cost model of Eq. 3: T(s) = a2 s^2 + a1 s + a0 with integer coefficients (the
    caller fits them to this library's kernel timings and rounds).  A long sequence costs each of
    its D ranks floor(T(s) / D); a bin costs its rank the sum of T over its sequences.
B2  line 4 "sort B by sequence length in descending order": the groups are sorted by the time
    they cost one rank, descending (ties: more ranks first, then the order Algorithm 1 made them).
B3  line 5 "divide B into buckets such that each bucket has an approximately equal sum of FLOPs":
    with n_buckets given, group g of the sorted list goes to bucket
    floor(n_buckets * (work of the groups before g) / (total work)), work = time x ranks (a
    group of zero work behind all the work stays in the last bucket).
B4  lines 7-9: max_time = max(exec_times); target ranks = {i : max_time - exec_times[i] > delta}.
    When no rank lags by more than delta (first of all at the start, all times 0) a new time
    step begins and every rank is a target.
B5  lines 10-17, DP-Balance: the next group of the first bucket goes to the D target ranks with
    the smallest exec_times (ties: lowest rank); when fewer than D ranks are targets, the least
    loaded other ranks fill up.  The D ranks start together (they exchange K/V) at the largest
    of their exec_times and all finish `time` later.  CP rank j is the j-th chosen rank in
    ascending rank order.  Targets are recomputed after every assignment (line 17).
B6  lines 18-20: an empty bucket is removed.

Under B4/B5 the target set is always a prefix of the ranks ordered by exec_time, so the ranks
chosen are the D least loaded ones whatever delta and the bucket boundaries are: DP-Balance is
longest-first list scheduling of gangs (tests/test_balance.py checks this equivalence, and
Graham's (4/3 - 1/(3m)) bound against brute force for D = 1).  delta and the buckets only matter
for PP-Balance, which is out of scope (no pipeline here).
"""
from .assign import groups


def seq_time(s, cost):
    a2, a1, a0 = cost
    return a2 * s * s + a1 * s + a0


def balance(lens, capacity, d_hdp, cost, n_buckets=4, delta=0):
    """Returns {"exec_times": [d_hdp], "makespan", "microbatches": [(rank, start, end, [(len, cp,
    cp_rank, input index), ...]), ...]} with the micro-batches sorted by (rank, start)."""
    if n_buckets < 1 or delta < 0 or any(c < 0 for c in cost):
        raise ValueError("bad argument")
    d, long_list, bins = groups(lens, capacity, d_hdp)
    # the groups with their per-rank time (B1)
    items = []
    for i in long_list:
        items.append({"ranks": d[i], "time": seq_time(lens[i], cost) // d[i], "seqs": [i]})
    for subset in bins:
        items.append({"ranks": 1, "time": sum(seq_time(lens[i], cost) for i in subset),
                      "seqs": subset})
    # lines 1-2
    micro_batches = []
    exec_times = [0] * d_hdp
    # lines 3-5: sort and bucketize (B2, B3)
    order = sorted(range(len(items)), key=lambda g: (-items[g]["time"], -items[g]["ranks"], g))
    total = sum(items[g]["time"] * items[g]["ranks"] for g in order)
    buckets = [[] for _ in range(n_buckets)]
    before = 0
    for g in order:
        b = min(n_buckets - 1, (n_buckets * before) // total) if total > 0 else 0
        buckets[b].append(g)
        before += items[g]["time"] * items[g]["ranks"]
    buckets = [b for b in buckets if b]
    # line 6
    while buckets:
        # lines 7-9 (B4)
        max_time = max(exec_times)
        targets = [i for i in range(d_hdp) if max_time - exec_times[i] > delta]
        if not targets:
            targets = list(range(d_hdp))
        # lines 10-17 (B5): one group per pass; line 17 recomputes the targets at the loop head
        g = buckets[0].pop(0)
        need = items[g]["ranks"]
        chosen = sorted(targets, key=lambda i: (exec_times[i], i))[:need]
        if len(chosen) < need:
            others = sorted((i for i in range(d_hdp) if i not in targets),
                            key=lambda i: (exec_times[i], i))
            chosen += others[:need - len(chosen)]
        chosen.sort()
        start = max(exec_times[i] for i in chosen)
        end = start + items[g]["time"]
        for j, i in enumerate(chosen):
            exec_times[i] = end
            if need > 1:
                s = items[g]["seqs"][0]
                micro_batches.append((i, start, end, [(lens[s], need, j, s)]))
            else:
                micro_batches.append((i, start, end, [(lens[s], 1, 0, s) for s in items[g]["seqs"]]))
        # lines 18-20 (B6)
        if not buckets[0]:
            buckets.pop(0)
    micro_batches.sort(key=lambda m: (m[0], m[1]))
    return {"exec_times": exec_times, "makespan": max(exec_times) if exec_times else 0,
            "microbatches": micro_batches}


def naive_times(lens, capacity, d_hdp, cost):
    """Per-rank time of Algorithm 1's own line 10 (oracle/assign.py) under the same cost model:
    a rank's time is the sum over its micro-batches (no barrier between rounds is modelled)."""
    from .assign import assign
    a = assign(lens, capacity, d_hdp)
    t = [0] * d_hdp
    for _, rank, seqs in a["microbatches"]:
        if seqs[0][1] > 1:
            t[rank] += seq_time(seqs[0][0], cost) // seqs[0][1]
        else:
            t[rank] += sum(seq_time(s[0], cost) for s in seqs)
    return t
