"""-m gpu: the bs_assign replay (paper_2502_21231_b200/replay.py) runs every micro-batch of a
small global batch through the C-ABI calls and reports a consistent per-rank picture."""
import pytest

pytestmark = pytest.mark.gpu

from paper_2502_21231_b200 import binding as B  # noqa: E402
from paper_2502_21231_b200 import replay as RP  # noqa: E402


def test_replay_of_a_small_global_batch():
    cap, d_hdp = 512, 4
    lens = RP.global_batch(3, 12, cap, (3, 2))
    assert sorted(lens)[-2:] == [2 * cap, 3 * cap] and len(lens) == 14
    a = B.assign(lens, cap, d_hdp)
    r = RP.replay(lens, cap, d_hdp, 4, 2, 64, seed=3)
    assert r["n_rounds"] == a["n_rounds"] and r["n_microbatches"] == len(a["microbatches"])
    assert len(r["rank_ms"]) == d_hdp and r["ranks_needed_max"] == 3
    busy = {rank for _, rank, _ in a["microbatches"]}
    for rank, ms in enumerate(r["rank_ms"]):
        assert (ms > 0) == (rank in busy)
    assert r["min_ms"] <= r["mean_ms"] <= r["max_ms"] and 0.0 <= r["idle_frac"] < 1.0
    assert r["tflops"] > 0


def test_balanced_replay_of_a_small_global_batch():
    cap, d_hdp = 512, 4
    lens = RP.global_batch(3, 24, cap, (3, 2))
    r = RP.replay_balanced(lens, cap, d_hdp, 4, 2, 64, seed=3)
    assert len(r["cost_fs"]) == 3 and all(c >= 0 for c in r["cost_fs"]) and sum(r["cost_fs"]) > 0
    bal = B.balance(lens, cap, d_hdp, r["cost_fs"])
    assert r["n_microbatches"] == len(bal["microbatches"])
    assert abs(r["model"]["balance_makespan_ms"] - bal["makespan"] * 1e-12) < 1e-3
    assert r["model"]["balance_makespan_ms"] <= r["model"]["naive_makespan_ms"] + 1e-9
    m = r["measured"]
    assert len(m["rank_finish_ms"]) == d_hdp and m["min_ms"] <= m["max_ms"]
    assert 0.0 <= m["idle_frac"] < 1.0


def test_static_cp_baseline_and_offload_probe():
    cap, d_hdp = 512, 4
    lens = RP.global_batch(3, 24, cap, (3, 2))
    r = RP.static_cp_baseline(lens, cap, 4, d_hdp, 4, 2, 64, seed=3)
    assert r["cp"] == 4 and r["groups"] == 1 and r["rank_ms"] > 0
    assert r["n_packed_sequences"] >= -(-sum(lens) // (4 * cap))
    o = RP.offload_probe((1024, 4096), 4, 2, 64, seed=3)
    assert [x["tokens"] for x in o] == [1024, 4096]
    for x in o:
        assert x["compute_ms"] > 0 and x["copy_ms"] > 0 and x["both_ms"] > 0
        assert x["bytes_each_way"] == x["tokens"] * (2 * 4 + 2 * 2) * 64 * 2
