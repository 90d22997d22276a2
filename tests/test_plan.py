"""bs_plan: the oracle planner (oracle/plan.py) pinned by brute force, PAPER.md:318's balance
statements and the golden worked examples; the library planner (csrc/plan.cpp through the C-ABI)
compared bit-exactly with the oracle planner.  CPU only (bs_plan is host code)."""
import os

import numpy as np
import pytest

import oracle
from oracle.plan import parts_of

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "plan_examples.txt")


def load_golden():
    examples, cur = [], None
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        head, body = line.split(":")
        tok = head.split()
        if tok[0] == "example":
            cur = dict(name=tok[1], seqs=[tuple(int(x) for x in s.split(",")) for s in body.split()],
                       steps=[])
            examples.append(cur)
        else:
            segs = [tuple(int(x) for x in s.split()) for s in body.split(";")]
            cur["steps"].append(dict(step=int(tok[1]), kv_rows=int(tok[3]), pairs=int(tok[5]),
                                     segs=segs))
    return examples


def lib_plan(seqs):
    from paper_2502_21231_b200 import binding
    return binding.plan(seqs)


PLANNERS = [pytest.param(oracle.oracle_plan, id="oracle"), pytest.param(lib_plan, id="library")]


@pytest.mark.parametrize("planner", PLANNERS)
@pytest.mark.parametrize("ex", load_golden(), ids=lambda e: e["name"])
def test_golden_examples(planner, ex):
    pl = planner(ex["seqs"])
    assert pl["n_steps"] == len(ex["steps"])
    for st, want in zip(pl["steps"], ex["steps"]):
        assert st["step"] == want["step"]
        assert st["kv_rows"] == want["kv_rows"]
        assert [tuple(s[:5]) for s in st["segs"]] == want["segs"]
        assert st["visible_pairs"] == want["pairs"]


@pytest.mark.parametrize("planner", PLANNERS)
def test_cfg5_formulae(planner):
    # L=2097152, cp=64, r=32, c=16384
    c = 16384
    pl = planner([(2097152, 64, 32)])
    assert pl["q_rows"] == 2 * c and pl["n_steps"] == 64
    total = 0
    for s, st in enumerate(pl["steps"]):
        segs = [tuple(x[:5]) for x in st["segs"]]
        if s == 0:
            assert segs == [(0, c, 0, c, 0), (c, 2 * c, 0, c, 1032192), (c, 2 * c, c, 2 * c, 0)]
        elif s <= 32:
            assert segs == [(0, c, 0, c, s * c), (c, 2 * c, 0, c, (63 + s) * c)]
        else:
            assert segs == [(c, 2 * c, 0, c, (s - 1) * c), (c, 2 * c, c, 2 * c, (64 - s) * c)]
        assert st["kv_rows"] == 2 * c and st["kv_src_rank"] == [(32 - s) % 64]
        assert st["visible_pairs"] == 536870912 + (c if s == 0 else 0)
        total += st["visible_pairs"]
    assert total == 34359754752


def visible_set(pl):
    """All (seq, q_pos, k_pos) triples a plan makes visible, enumerated pair by pair from the
    segment descriptors and the row->(seq,pos) maps; with multiplicity."""
    out = []
    for st in pl["steps"]:
        for (q0, q1, k0, k1, off, sq) in st["segs"]:
            for a in range(q1 - q0):
                for b in range(k1 - k0):
                    if b <= a + off:
                        assert pl["q_seq"][q0 + a] == sq == st["k_seq"][k0 + b]
                        out.append((sq, int(pl["q_pos"][q0 + a]), int(st["k_pos"][k0 + b])))
    return out


@pytest.mark.parametrize("L,N", [(64, 4), (50, 4), (7, 4), (96, 3), (5, 8), (33, 2), (1, 2)])
def test_union_over_ranks_is_causal_set_exactly_once(L, N):
    """the N ranks together compute exactly causal attention of the sequence."""
    seen = []
    rows = 0
    for r in range(N):
        pl = oracle.oracle_plan([(L, N, r)])
        rows += pl["q_rows"]
        seen += visible_set(pl)
        assert sum(st["visible_pairs"] for st in pl["steps"]) == len(visible_set(pl))
    assert rows == L
    want = sorted((0, i, j) for i in range(L) for j in range(i + 1))
    assert sorted(seen) == want


@pytest.mark.parametrize("L,N", [(64, 4), (96, 3), (4096, 8), (1024, 64)])
def test_balance_statements_divisible(L, N):
    """'each device holds 1/N of all the subsequences and covers 1/N of the attention mask area
    ... the same data exchange volume', divisible case: L/N rows per rank, equal
    KV rows per step, 2c^2 pairs per step (+c at step 0), total L(L+1)/2N."""
    c = L // (2 * N)
    for r in range(N):
        pl = oracle.oracle_plan([(L, N, r)])
        assert pl["q_rows"] == L // N
        tot = 0
        for s, st in enumerate(pl["steps"]):
            assert st["kv_rows"] == 2 * c
            assert st["visible_pairs"] == 2 * c * c + (c if s == 0 else 0)
            assert st["kv_src_rank"] == [(r - s) % N]
            tot += st["visible_pairs"]
        assert tot * N == L * (L + 1) // 2


def test_parts_tile_sequence_and_ragged_balance():
    for L in (1, 5, 7, 50, 97, 1000):
        for N in (2, 3, 4, 8):
            ps = parts_of(L, N)
            assert ps[0][0] == 0 and ps[-1][1] == L
            assert all(a[1] == b[0] for a, b in zip(ps, ps[1:]))
            sizes = [e - b for b, e in ps]
            assert max(sizes) - min(sizes) <= 1
            for r in range(N):
                assert abs(oracle.oracle_plan([(L, N, r)])["q_rows"] - L / N) <= 2


def test_mixed_plan_structure():
    seqs = [(50, 4, 1), (7, 1, 0), (12, 2, 0), (3, 8, 5)]
    pl = oracle.oracle_plan(seqs)
    assert pl["n_steps"] == 8
    assert pl["cu_rows_q"][0] == 0 and pl["cu_rows_q"][-1] == pl["q_rows"] == len(pl["q_pos"])
    # step 0's KV layout is the Q layout (the device's own K/V)
    st0 = pl["steps"][0]
    assert st0["kv_rows"] == pl["q_rows"]
    assert np.array_equal(st0["k_seq"], pl["q_seq"]) and np.array_equal(st0["k_pos"], pl["q_pos"])
    # two segments of a step have identical or disjoint q ranges, at most two per q range
    for st in pl["steps"]:
        qr = [(s[0], s[1]) for s in st["segs"]]
        for a in qr:
            for b in qr:
                assert a == b or a[1] <= b[0] or b[1] <= a[0]
            assert qr.count(a) <= 2
    # every visible pair obeys the definition on global positions, and every real row sees
    # itself exactly once over all steps
    vs = visible_set(pl)
    assert all(k <= q for _, q, k in vs)
    self_pairs = [(s, q) for s, q, k in vs if q == k]
    assert sorted(self_pairs) == sorted(zip(pl["q_seq"].tolist(), pl["q_pos"].tolist()))


@pytest.mark.parametrize("seed", range(6))
def test_library_plan_bit_exact_vs_oracle(seed):
    rng = np.random.default_rng(seed)
    seqs = []
    for _ in range(int(rng.integers(1, 12))):
        cp = int(rng.choice([1, 1, 1, 2, 3, 4, 8, 16]))
        L = int(rng.integers(1, 3000))
        seqs.append((L, cp, int(rng.integers(0, cp))))
    a, b = oracle.oracle_plan(seqs), lib_plan(seqs)
    assert a["q_rows"] == b["q_rows"] and a["n_steps"] == b["n_steps"]
    assert list(a["cu_rows_q"]) == list(b["cu_rows_q"])
    assert np.array_equal(a["q_seq"], b["q_seq"]) and np.array_equal(a["q_pos"], b["q_pos"])
    for sa, sb in zip(a["steps"], b["steps"]):
        assert [tuple(x) for x in sa["segs"]] == [tuple(x) for x in sb["segs"]]
        for k in ("step", "kv_rows", "visible_pairs"):
            assert sa[k] == sb[k], k
        for k in ("kv_seq", "kv_src_rank", "cu_rows_k"):
            assert list(sa[k]) == list(sb[k]), k
        assert np.array_equal(sa["k_seq"], sb["k_seq"]) and np.array_equal(sa["k_pos"], sb["k_pos"])


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_library_plan_bit_exact_on_configs(cfg):
    from paper_2502_21231_b200.synth import make_workload
    w = make_workload(cfg)
    a, b = oracle.oracle_plan(w.seqs), lib_plan(w.seqs)
    assert a["q_rows"] == b["q_rows"] and a["n_steps"] == b["n_steps"]
    assert np.array_equal(a["q_pos"], b["q_pos"]) and np.array_equal(a["q_seq"], b["q_seq"])
    for sa, sb in zip(a["steps"], b["steps"]):
        assert [tuple(x) for x in sa["segs"]] == [tuple(x) for x in sb["segs"]]
        assert sa["visible_pairs"] == sb["visible_pairs"] and sa["kv_rows"] == sb["kv_rows"]
        assert np.array_equal(sa["k_pos"], sb["k_pos"])


def _same_plan(a, b):
    assert a["q_rows"] == b["q_rows"] and a["n_steps"] == b["n_steps"]
    assert list(a["cu_rows_q"]) == list(b["cu_rows_q"])
    assert np.array_equal(a["q_seq"], b["q_seq"]) and np.array_equal(a["q_pos"], b["q_pos"])
    for sa, sb in zip(a["steps"], b["steps"]):
        assert [tuple(x) for x in sa["segs"]] == [tuple(x) for x in sb["segs"]]
        for k in ("step", "kv_rows", "visible_pairs"):
            assert sa[k] == sb[k], k
        for k in ("kv_seq", "kv_src_rank", "cu_rows_k"):
            assert list(sa[k]) == list(sb[k]), k
        assert np.array_equal(sa["k_seq"], sb["k_seq"]) and np.array_equal(sa["k_pos"], sb["k_pos"])


@pytest.mark.parametrize("seed", range(4))
def test_plan_uniform_matches_oracle(seed):
    """bs_plan_uniform (north_star: "per-sequence lengths and a CP degree"): sequences of at least
    min_shard_len tokens get (cp, rank), the rest stay whole - the data-aware sharding rule of
    PAPER.md:165 - and the result is bs_plan's on that list, compared with the oracle planner."""
    from paper_2502_21231_b200 import binding
    rng = np.random.default_rng(100 + seed)
    lens = [int(x) for x in rng.integers(1, 4000, int(rng.integers(1, 15)))]
    cp = int(rng.choice([1, 2, 4, 8]))
    rank = int(rng.integers(0, cp))
    min_len = int(rng.choice([1, 512, 2048, 5000]))
    seqs = [(L, cp, rank) if L >= min_len else (L, 1, 0) for L in lens]
    _same_plan(oracle.oracle_plan(seqs), binding.plan_uniform(lens, cp, rank, min_len))
    with pytest.raises(binding.BsError):
        binding.plan_uniform(lens, cp, cp, min_len)   # rank outside [0, cp)


def test_library_plan_errors():
    from paper_2502_21231_b200 import binding
    for bad in ([(0, 1, 0)], [(5, 0, 0)], [(5, 2, 2)], [(5, 2, -1)]):
        with pytest.raises(binding.BsError):
            binding.plan(bad)
    assert binding.plan([])["n_steps"] == 0
