"""not gpu: `bs_balance` (Algorithm 2, DP-Balance).  The oracle (oracle/balance.py)
against what pins it - a batch worked by hand, validity and lower bounds on random batches,
invariance under delta and the bucket count (readings B4/B5), Graham's list-scheduling bound
against brute force - and the library's bs_balance against the oracle, bit-exact."""
import itertools
import random

import pytest

import oracle.assign as OA
import oracle.balance as OB


def lib_balance(lens, capacity, d_hdp, cost, n_buckets=4, delta=0):
    from paper_2502_21231_b200 import binding as B
    return B.balance(lens, capacity, d_hdp, cost, n_buckets, delta)


IMPLS = [pytest.param(OB.balance, id="oracle"), pytest.param(lib_balance, id="library")]


@pytest.mark.parametrize("impl", IMPLS)
def test_hand_worked(impl):
    # T(s) = s^2, capacity 10, 4 ranks.  Groups: 25 on 3 ranks (625 // 3 = 208 each), 15 on 2 ranks
    # (225 // 2 = 112 each), bins {8} (64) and {7, 3} (49 + 9 = 58); that is also the sorted order.
    # 25 -> ranks 0,1,2 at 0..208.  15 needs two ranks: only rank 3 lags (by 208), the least loaded
    # other rank is 0; they start together at 208 -> 320.  {8}: ranks 1, 2 lag, rank 1 first:
    # 208..272.  {7,3}: rank 2 is the least loaded: 208..266.
    a = impl([25, 15, 8, 7, 3], 10, 4, (1, 0, 0))
    assert a["exec_times"] == [320, 272, 266, 320] and a["makespan"] == 320
    assert a["microbatches"] == [
        (0, 0, 208, [(25, 3, 0, 0)]), (0, 208, 320, [(15, 2, 0, 1)]),
        (1, 0, 208, [(25, 3, 1, 0)]), (1, 208, 272, [(8, 1, 0, 2)]),
        (2, 0, 208, [(25, 3, 2, 0)]), (2, 208, 266, [(7, 1, 0, 3), (3, 1, 0, 4)]),
        (3, 208, 320, [(15, 2, 1, 1)])]


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("n_buckets", [1, 2, 4, 9])
def test_zero_work_group_stays_in_the_last_bucket(impl, n_buckets):
    """Reading B3's corner: T(s) = 1 for every sequence, so a long sequence on D = 2 ranks costs
    each rank floor(1 / 2) = 0 - a group of zero work, sorted behind all the work.  Its bucket
    index floor(n_buckets * work before / total work) would be n_buckets: it stays in the last
    bucket (B3) instead of indexing past the end.  Worked by hand: bin {5, 5} costs 2 and goes to
    rank 0 at 0..2; the long group then goes to the two least loaded ranks that lag (1 and 2),
    starting at 0 and ending at 0."""
    a = impl([20, 5, 5], 10, 4, (0, 0, 1), n_buckets, 0)
    assert a["exec_times"] == [2, 0, 0, 0] and a["makespan"] == 2
    assert a["microbatches"] == [(0, 0, 2, [(5, 1, 0, 1), (5, 1, 0, 2)]),
                                 (1, 0, 0, [(20, 2, 0, 0)]), (2, 0, 0, [(20, 2, 1, 0)])]
    # all work zero (total work 0): everything goes to bucket 0 and is still scheduled once
    b = impl([20, 5, 5], 10, 4, (0, 0, 0), n_buckets, 0)
    assert b["makespan"] == 0 and len(b["microbatches"]) == 3


def random_batch(g):
    cap = g.choice([4, 10, 100, 8192])
    d_hdp = g.choice([1, 2, 3, 8, 32])
    n = g.randrange(1, 40)
    lens = [min(max(1, int(g.lognormvariate(0, 1.4) * cap / 3)), cap * d_hdp) for _ in range(n)]
    cost = (g.choice([0, 1, 3]), g.choice([0, 1, 50]), g.choice([0, 7]))
    return lens, cap, d_hdp, cost


@pytest.mark.parametrize("impl", IMPLS)
def test_validity_and_lower_bounds(impl):
    g = random.Random(11)
    for _ in range(150):
        lens, cap, d_hdp, cost = random_batch(g)
        a = impl(lens, cap, d_hdp, cost, g.choice([1, 2, 4, 9]), g.choice([0, 5, 1000]))
        d, long_list, bins = OA.groups(lens, cap, d_hdp)
        seen, shards, work = set(), {}, 0
        per_rank = {}
        for rank, start, end, seqs in a["microbatches"]:
            assert 0 <= rank < d_hdp and 0 <= start <= end
            per_rank.setdefault(rank, []).append((start, end))
            if seqs[0][1] > 1:
                length, cp, j, i = seqs[0]
                assert len(seqs) == 1 and cp == d[i] and length == lens[i]
                assert end - start == OB.seq_time(length, cost) // cp
                shards.setdefault(i, []).append((rank, start, end, j))
            else:
                assert sum(s[0] for s in seqs) <= cap
                assert end - start == sum(OB.seq_time(s[0], cost) for s in seqs)
                for s in seqs:
                    assert s[3] not in seen and d[s[3]] == 1
                    seen.add(s[3])
            work += end - start
        for i in long_list:   # the D ranks of a long sequence run it at the same time
            sh = sorted(shards[i], key=lambda x: x[3])
            assert [x[3] for x in sh] == list(range(d[i])) and len({x[0] for x in sh}) == d[i]
            assert len({(x[1], x[2]) for x in sh}) == 1
            assert [x[0] for x in sh] == sorted(x[0] for x in sh)
        assert seen == {i for i in range(len(lens)) if d[i] == 1}
        for rank in range(d_hdp):   # a rank runs one micro-batch at a time
            spans = sorted(per_rank.get(rank, []))
            for (s0, e0), (s1, e1) in zip(spans, spans[1:]):
                assert e0 <= s1
            assert a["exec_times"][rank] == (max(e for _, e in spans) if spans else 0)
        assert a["makespan"] == max(a["exec_times"])
        longest = max([e - s for _, s, e, _ in a["microbatches"]], default=0)
        assert a["makespan"] >= max(longest, -(-work // d_hdp))


def test_delta_and_buckets_do_not_change_dp_balance():
    """Readings B4/B5: the targets are a prefix of the ranks ordered by exec_time."""
    g = random.Random(5)
    for _ in range(100):
        lens, cap, d_hdp, cost = random_batch(g)
        ref = OB.balance(lens, cap, d_hdp, cost, 1, 0)
        for nb, delta in ((3, 0), (7, 13), (2, 10 ** 9)):
            assert OB.balance(lens, cap, d_hdp, cost, nb, delta) == ref


def test_graham_bound_against_brute_force():
    """With one rank per group DP-Balance is longest-processing-time-first list scheduling:
    makespan <= (4/3 - 1/(3m)) OPT (Graham 1969).  OPT by exhaustive assignment."""
    g = random.Random(3)
    for _ in range(60):
        m = g.choice([2, 3])
        cap = 10
        lens = [g.randrange(6, 11) for _ in range(g.randrange(2, 8))]   # no two fit one bin
        cost = (g.choice([1, 2]), g.choice([0, 3]), 0)
        a = OB.balance(lens, cap, m, cost)
        jobs = [OB.seq_time(s, cost) for s in lens]
        opt = min(max(sum(j for j, r in zip(jobs, asg) if r == k) for k in range(m))
                  for asg in itertools.product(range(m), repeat=len(jobs)))
        assert opt <= a["makespan"] and 3 * m * a["makespan"] <= (4 * m - 1) * opt


def test_balance_is_not_worse_than_naive_on_long_tailed_batches():
    g = random.Random(8)
    wins = 0
    for _ in range(40):
        cap, d_hdp = 8192, 16
        lens = [min(max(64, int(g.lognormvariate(7, 1.2))), cap) for _ in range(96)]
        lens += [cap * m for m in (8, 4, 2, 2)]
        g.shuffle(lens)
        cost = (1, 4000, 0)
        bal = OB.balance(lens, cap, d_hdp, cost)["makespan"]
        naive = max(OB.naive_times(lens, cap, d_hdp, cost))
        assert bal <= naive
        wins += bal < naive
    assert wins >= 30


def test_library_matches_oracle_bit_exact():
    g = random.Random(17)
    for _ in range(300):
        lens, cap, d_hdp, cost = random_batch(g)
        nb, delta = g.choice([1, 4, 16]), g.choice([0, 9, 10 ** 6])
        assert lib_balance(lens, cap, d_hdp, cost, nb, delta) == OB.balance(lens, cap, d_hdp, cost, nb, delta)
