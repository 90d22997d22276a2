"""-m gpu: seeded random HDP buffers through the whole path (forward of every ring step, merge,
prep, backward of every ring step, finish) against the fp64 oracle, every element.

Each case draws what a rank's micro-batch can look like (whole short sequences
next to zigzag shards of long ones): 1-7 sequences, lengths from 1 token to a few
tiles with ragged ends, CP degrees 1-8 with a random rank, GQA group sizes 1-8 (3 and 5 included,
which no config uses), D = 64 or 128, the accumulator cleared by prep or by the first forward.
The point is the combinations no hand-written case lists: a lone first tile next to a one-token
document, a range that ends one row into a tile, a shard whose low part sees nothing in a step."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2502_21231_b200.synth.workloads import Workload  # noqa: E402


def _draw(seed):
    g = np.random.default_rng(1000 + seed)
    group = int(g.choice([1, 1, 2, 3, 4, 5, 6, 8]))
    hkv = int(g.choice([1, 2, 3]))
    D = int(g.choice([64, 128, 128]))
    seqs, rows = [], 0
    for _ in range(int(g.integers(1, 8))):
        cp = int(g.choice([1, 1, 1, 2, 3, 4, 8]))
        kind = g.integers(0, 4)
        if kind == 0:
            L = int(g.integers(1, 40))                      # a few tokens
        elif kind == 1:
            L = int(g.integers(1, 6)) * 128 + int(g.choice([-1, 0, 1]))   # next to a tile boundary
        else:
            L = int(g.integers(40, 900))
        L = max(1, L) * (cp if cp > 1 and g.integers(0, 2) else 1)        # longer when sharded
        seqs.append((L, cp, int(g.integers(0, cp))))
        rows += -(-L // cp)
        if rows > 2600:
            break
    return Workload(f"fuzz{seed}", group * hkv, hkv, D, seqs, 4000 + seed), bool(g.integers(0, 2))


@pytest.mark.parametrize("seed", range(24))
def test_random_hdp_buffer(seed):
    import gpu_util as U
    w, fused_clear = _draw(seed)
    print(f"{w.name}: heads {w.n_q_heads}/{w.n_kv_heads}, D {w.head_dim}, seqs {w.seqs}, "
          f"accumulator cleared by the {'forward' if fused_clear else 'prep'}")
    run = U.DeviceRun(w, fused_clear=fused_clear)
    O, LSE, _ = run.forward()
    U.check_forward(run, O, LSE, label=f"{w.name}: ")
    dQ, grads, _ = run.backward(O, LSE)
    U.check_backward(run, dQ, grads, O, LSE, label=f"{w.name}: ")
