"""-m gpu: forward + merge + backward (prep, bs_attn_bwd per step, finish) through the C-ABI
against the fp64 oracle over all keys: every element of O, LSE, dQ, dK, dV on small packed /
zigzag-CP workloads and on scaled-down twins of configs 3-5 (same N, group size, D and segment
pattern).  Gradients are compared whole, per (ring step, document, 128-row
chunk) x head block, and element by element (gpu_util.grad_compare)."""
import pytest

pytestmark = pytest.mark.gpu

from paper_2502_21231_b200.synth import workloads  # noqa: E402
from paper_2502_21231_b200.synth.workloads import Workload  # noqa: E402


def _run(w, fused_clear=False):
    import gpu_util as U
    run = U.DeviceRun(w, fused_clear=fused_clear)
    O, LSE, _ = run.forward()
    U.check_forward(run, O, LSE, label=f"{w.name}: ")
    dQ, grads, _ = run.backward(O, LSE)
    return U.check_backward(run, dQ, grads, O, LSE, label=f"{w.name}: ")


@pytest.mark.parametrize("lens,Hq,Hkv,D", [
    ([1], 1, 1, 64), ([64], 1, 1, 128), ([128], 2, 2, 128), ([129, 255, 257], 4, 2, 128),
    ([700], 2, 1, 128), ([300, 77, 1, 513, 64], 4, 4, 64), ([1100, 5], 8, 2, 128),
    ([130, 2, 391], 6, 1, 128), ([1, 640, 3], 8, 1, 128), ([257, 100], 16, 2, 64)])
def test_packed_documents(lens, Hq, Hkv, D):
    print(_run(Workload("packed", Hq, Hkv, D, [(L, 1, 0) for L in lens], 78)))


@pytest.mark.parametrize("L,N,r", [(2048, 4, 0), (2048, 4, 1), (2048, 4, 3), (1999, 4, 2),
                                    (50, 4, 1), (3000, 3, 1)])
def test_zigzag_cp(L, N, r):
    print(_run(Workload("cp", 4, 2, 128, [(L, N, r)], 92 + r)))


def test_mixed_hdp_buffer():
    print(_run(Workload("mixed", 4, 1, 128, [(50, 4, 1), (7, 1, 0), (1200, 2, 0), (300, 1, 0)], 6)))


# Scaled-down twins of configs 3-5 (GQA PAPER.md:316, zigzag PAPER.md:318): part
# length 256 and a ragged twin (2N does not divide L, parts unaligned to any tile), full tensors.
# The group size Hq/Hkv is the config's (8, 4, 6); two KV groups keep the oracle pass in seconds.
@pytest.mark.parametrize("ragged", [False, True], ids=["c256", "ragged"])
@pytest.mark.parametrize("r", range(8))
def test_twin_of_cfg3_every_rank(r, ragged):
    print(_run(workloads.scaled_twin(3, 256, ragged, rank=r, kv_heads=2)))


@pytest.mark.parametrize("ragged", [False, True], ids=["c256", "ragged"])
@pytest.mark.parametrize("r", range(4))
def test_twin_of_cfg4_every_rank(r, ragged):
    print(_run(workloads.scaled_twin(4, 256, ragged, rank=r, kv_heads=2), fused_clear=(r == 1)))


@pytest.mark.parametrize("ragged", [False, True], ids=["c256", "ragged"])
@pytest.mark.parametrize("r", [0, 31, 32, 63])
def test_twin_of_cfg5_ranks(r, ragged):
    # (one KV group of 6 query heads: the oracle pass over 32768 keys stays at ~6 s per case)
    print(_run(workloads.scaled_twin(5, 256, ragged, rank=r, kv_heads=1)))


def test_twin_of_cfg3_all_eight_groups():
    """The config's own head counts (64 / 8) once, at part length 128."""
    print(_run(workloads.scaled_twin(3, 128, False, rank=0)))


@pytest.mark.parametrize("seqs,Hq,Hkv,D", [
    ([(129, 1, 0), (255, 1, 0), (257, 1, 0)], 4, 2, 128),       # ragged units overhang into the next document
    ([(300, 1, 0), (77, 1, 0), (1, 1, 0), (513, 1, 0)], 4, 4, 64),
    ([(2048, 4, 1)], 4, 2, 128),                                # low part rows see nothing in some steps
    ([(50, 4, 1), (7, 1, 0), (1200, 2, 0), (300, 1, 0)], 4, 1, 128)])
def test_accumulator_cleared_by_forward(seqs, Hq, Hkv, D):
    """dQ_acc (NaN-filled) is cleared by the first step's bs_attn_fwd, prep gets dQ_acc = NULL."""
    print(_run(Workload("fused", Hq, Hkv, D, seqs, 93), fused_clear=True))


def test_static_cp_micro_batch():
    """The static-CP packed baseline (Fig. 14 at PAPER.md:306-308): EVERY
    document of a packed sequence is cut 2 x 16 ways, so a rank holds parts of 10-50 rows and a
    call has dozens of segments per 128-row tile.  Same kernels, other bs_plan inputs."""
    import numpy as np
    g = np.random.default_rng(14)
    lens = [int(x) for x in g.integers(330, 1600, 30)]
    for r in (0, 9):
        print(_run(Workload(f"static_cp_r{r}", 8, 2, 128, [(L, 16, r) for L in lens], 140 + r)))
