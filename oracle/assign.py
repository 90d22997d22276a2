"""TEST INFRASTRUCTURE ONLY: oracle of `bs_assign`, the naive HDP solution (Algorithm 1,
lines 214-235, routine described at PAPER.md:262) with offload ratio r = 0.

Plain Python, integers only, written in the order of the algorithm's lines.  Pinned by the rank
counts the paper prints (tests/golden/assign_examples.txt) and by brute force on tiny batches
(tests/test_assign.py).  Readings of the points the paper leaves open are the ones DESIGN.md
section 11 lists (R1-R4 below).

R1  D(s) (Eq. 3) with r = 0 and Act(s) = alpha2 * s (beta2 = 0):
    D(s) = ceil((2 Act(s) + (l - 2) Act(s)) / (l Act(C))) = ceil(s / C).
R2  "if d_i == 0 ... add s_i to pack_list" (lines 3-4, garbled): a sequence that needs no
    partitioning, D(s_i) = 1, is packed; every other one keeps map_d[s_i] = D(s_i).
R3  lines 7-9, "while pack_list is not empty: pack subset by best-fit strategy to fill capacity
    C": one bin per loop iteration; the bin is filled by repeatedly taking the longest remaining
    sequence that still fits (ties: lowest input index) until none fits.
R4  line 10, "assign sequences to d_hdp HDP ranks based on map_d": a training step is a number of
    rounds; in a round every rank runs at most one micro-batch and the D(s_i) ranks of a long
    sequence run it in the same round (they exchange K/V).  Long sequences are placed in input
    order into the first round that still has D(s_i) free ranks, then the bins, in the order they
    were made, each into the first round with a free rank; inside a round ranks are handed out
    from 0 upwards in placement order (96 ranks for a 768K sequence and the other 32
    ranks for 32 x 8K sequences).  A sequence with D(s_i) > d_hdp does not fit: error.
"""


def ranks_needed(s, capacity):
    """D(s) of Eq. 3 with r = 0 (R1)."""
    return -(-s // capacity)


def groups(lens, capacity, d_hdp):
    """Lines 1-9 of Algorithm 1: (d, long_list, bins) - D(s_i) of every sequence, the indices of
    the long sequences in input order, the bins (lists of indices) in the order they are made."""
    if capacity < 1 or d_hdp < 1 or any(s < 1 for s in lens):
        raise ValueError("bad argument")
    # lines 1-6
    d = [ranks_needed(s, capacity) for s in lens]
    if any(x > d_hdp for x in d):
        raise ValueError("sequence needs more ranks than d_hdp")
    pack_list = [i for i in range(len(lens)) if d[i] == 1]
    long_list = [i for i in range(len(lens)) if d[i] > 1]
    # lines 7-9 (R3)
    bins = []
    while pack_list:
        room, subset = capacity, []
        while True:
            fit = [i for i in pack_list if lens[i] <= room]
            if not fit:
                break
            best = max(fit, key=lambda i: (lens[i], -i))
            subset.append(best)
            pack_list.remove(best)
            room -= lens[best]
        bins.append(subset)
    return d, long_list, bins


def assign(lens, capacity, d_hdp):
    """Returns {"d": [D(s_i)], "n_rounds": R, "microbatches": [(round, rank, [(len, cp, cp_rank,
    input index), ...]), ...]} with the micro-batches sorted by (round, rank)."""
    d, long_list, bins = groups(lens, capacity, d_hdp)
    # line 10 (R4)
    free = []          # free ranks of each round
    out = []
    def place(need):
        for k in range(len(free)):
            if free[k] >= need:
                break
        else:
            free.append(d_hdp)
            k = len(free) - 1
        first = d_hdp - free[k]
        free[k] -= need
        return k, first
    for i in long_list:
        k, first = place(d[i])
        for j in range(d[i]):
            out.append((k, first + j, [(lens[i], d[i], j, i)]))
    for subset in bins:
        k, first = place(1)
        out.append((k, first, [(lens[i], 1, 0, i) for i in subset]))
    out.sort(key=lambda m: (m[0], m[1]))
    return {"d": d, "n_rounds": len(free), "microbatches": out}
