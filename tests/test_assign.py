"""not gpu: `bs_assign` (naive HDP, Algorithm 1 with r = 0).  The oracle
(oracle/assign.py) against what pins it - the rank counts the paper prints
(tests/golden/assign_examples.txt), two batches worked by hand below, and invariants checked by
brute force on random batches - and the library's bs_assign (csrc/assign.cpp through the C-ABI)
against the oracle, bit-exact."""
import os
import random

import pytest

import oracle.assign as OA

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "assign_examples.txt")


def golden_lines(kind):
    out = []
    for line in open(GOLDEN):
        line = line.strip()
        if line.startswith(kind + " "):
            out.append(line[len(kind) + 1:])
    return out


def lib_assign(lens, capacity, d_hdp):
    from paper_2502_21231_b200 import binding as B
    return B.assign(lens, capacity, d_hdp)


IMPLS = [pytest.param(OA.assign, id="oracle"), pytest.param(lib_assign, id="library")]


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("line", golden_lines("ranks"))
def test_paper_rank_counts(impl, line):
    cap, length, d = (int(x) for x in line.split())
    a = impl([length], cap, 1024)
    assert a["d"] == [d]
    assert len(a["microbatches"]) == d and a["n_rounds"] == 1
    assert [m[1] for m in a["microbatches"]] == list(range(d))
    assert all(m[2] == [(length, d, j, 0)] for j, m in enumerate(a["microbatches"]))


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("line", golden_lines("round"))
def test_paper_round(impl, line):
    head, want = line.split("->")
    cfg, batch = head.split(":")
    cap, d_hdp = (int(x) for x in cfg.split())
    lens = []
    for tok in batch.split():
        length, count = tok.split("x")
        lens += [int(length)] * int(count)
    a = impl(lens, cap, d_hdp)
    assert a["n_rounds"] == 1
    by_rank = {m[1]: m[2] for m in a["microbatches"]}
    assert sorted(by_rank) == list(range(d_hdp))
    for tok in want.split():
        length, span = tok.split(":")
        lo, hi = (int(x) for x in span.split("-"))
        for r in range(lo, hi + 1):
            assert [s[0] for s in by_rank[r]] == [int(length)]


@pytest.mark.parametrize("impl", IMPLS)
def test_hand_worked_packing(impl):
    # capacity 8, all short.  Bin 1: longest 5 (room 3), longest that fits 3 - the first of the
    # two 3s - (room 0).  Bin 2: 4 (room 4), 3 (room 1), 1 (room 0).  Bin 3: 2, 2 (room 4; nothing
    # left).  One rank per bin, three ranks of round 0.
    a = impl([5, 4, 3, 3, 2, 2, 1], 8, 4)
    assert a["d"] == [1] * 7 and a["n_rounds"] == 1
    assert a["microbatches"] == [
        (0, 0, [(5, 1, 0, 0), (3, 1, 0, 2)]),
        (0, 1, [(4, 1, 0, 1), (3, 1, 0, 3), (1, 1, 0, 6)]),
        (0, 2, [(2, 1, 0, 4), (2, 1, 0, 5)])]


@pytest.mark.parametrize("impl", IMPLS)
def test_hand_worked_rounds(impl):
    # capacity 10, 4 ranks.  25 -> 3 ranks: round 0, ranks 0-2.  15 -> 2 ranks: round 0 has one
    # free rank, so round 1, ranks 0-1.  35 -> 4 ranks: round 2.  Bins: {8} (room 2: neither 7 nor
    # 3 fits), {7, 3}.  {8} -> round 0 rank 3; {7, 3} -> round 1 rank 2.
    a = impl([25, 15, 35, 8, 7, 3], 10, 4)
    assert a["d"] == [3, 2, 4, 1, 1, 1] and a["n_rounds"] == 3
    mb = a["microbatches"]
    assert mb[:4] == [(0, 0, [(25, 3, 0, 0)]), (0, 1, [(25, 3, 1, 0)]), (0, 2, [(25, 3, 2, 0)]),
                      (0, 3, [(8, 1, 0, 3)])]
    assert mb[4:7] == [(1, 0, [(15, 2, 0, 1)]), (1, 1, [(15, 2, 1, 1)]),
                       (1, 2, [(7, 1, 0, 4), (3, 1, 0, 5)])]
    assert mb[7:] == [(2, j, [(35, 4, j, 2)]) for j in range(4)]


@pytest.mark.parametrize("impl", IMPLS)
def test_invariants_on_random_batches(impl):
    g = random.Random(20250221)
    for _ in range(200):
        cap = g.choice([1, 3, 8, 100, 8192])
        d_hdp = g.choice([1, 2, 5, 16, 64])
        n = g.randrange(0, 40)
        lens = [max(1, int(g.lognormvariate(0, 1.5) * cap / 3)) for _ in range(n)]
        lens = [min(s, cap * d_hdp) for s in lens]
        a = impl(lens, cap, d_hdp)
        # D is the least number of capacity-C ranks that hold the sequence
        for s, d in zip(lens, a["d"]):
            assert (d - 1) * cap < s <= d * cap
        seen_slot, shards, packed, bins = set(), {}, {}, []
        for rnd, rank, seqs in a["microbatches"]:
            assert 0 <= rank < d_hdp and 0 <= rnd < a["n_rounds"]
            assert (rnd, rank) not in seen_slot
            seen_slot.add((rnd, rank))
            if seqs[0][1] > 1:   # one shard of a long sequence
                assert len(seqs) == 1
                length, cp, j, i = seqs[0]
                assert length == lens[i] and cp == a["d"][i]
                shards.setdefault(i, []).append((rnd, rank, j))
            else:                # a bin of whole sequences within the capacity
                assert all(s[1] == 1 and s[2] == 0 and s[0] == lens[s[3]] for s in seqs)
                assert sum(s[0] for s in seqs) <= cap
                for s in seqs:
                    assert s[3] not in packed
                    packed[s[3]] = len(bins)
                bins.append(seqs)
        # every sequence exactly once: as D shards in one round on D ranks, or in one bin
        for i, d in enumerate(a["d"]):
            if d > 1:
                assert i not in packed
                got = sorted(shards[i], key=lambda x: x[2])
                assert [x[2] for x in got] == list(range(d))
                assert len({x[0] for x in got}) == 1 and len({x[1] for x in got}) == d
            else:
                assert i in packed and i not in shards
        # R3: a bin is closed only when nothing that is left fits
        for b, seqs in enumerate(bins):
            room = cap - sum(s[0] for s in seqs)
            for later in bins[b + 1:]:
                assert all(s[0] > room for s in later)
            assert [s[0] for s in seqs] == sorted((s[0] for s in seqs), reverse=True)
        # R4: no earlier round could have taken a later micro-batch group
        used = [0] * a["n_rounds"]
        for rnd, rank, seqs in a["microbatches"]:
            used[rnd] += 1
        assert all(u >= 1 for u in used)


@pytest.mark.parametrize("impl", IMPLS)
def test_errors(impl):
    with pytest.raises(Exception):
        impl([100], 8, 4)       # needs 13 ranks, 4 exist
    with pytest.raises(Exception):
        impl([0, 5], 8, 4)
    with pytest.raises(Exception):
        impl([5], 0, 4)


def test_library_matches_oracle_bit_exact():
    g = random.Random(7)
    for _ in range(300):
        cap = g.choice([1, 2, 7, 64, 8192, 65536])
        d_hdp = g.choice([1, 3, 8, 128, 1024])
        n = g.randrange(0, 120)
        lens = [min(max(1, int(g.paretovariate(1.1) * cap / 4)), cap * d_hdp) for _ in range(n)]
        assert lib_assign(lens, cap, d_hdp) == OA.assign(lens, cap, d_hdp)
