"""-m gpu: bs_attn_fwd (+ bs_lse_merge) through the C-ABI against the fp64 oracle, every output
element, on cfg1 and on small packed / zigzag-CP workloads spanning several tiles and ragged
tails."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2502_21231_b200.synth import workloads  # noqa: E402
from paper_2502_21231_b200.synth.workloads import Workload  # noqa: E402


def _run(w, merge=True):
    import gpu_util as U
    run = U.DeviceRun(w)
    O, LSE, parts = run.forward(merge=merge)
    return U.check_forward(run, O, LSE), run, parts


def test_cfg1_tiny_packed_forward():
    (eo, el), run, _ = _run(workloads.make_workload(1))
    assert run.q_rows == 960
    print(f"cfg1: O max abs err {eo:.3e}, LSE abs err {el:.3e}")


@pytest.mark.parametrize("lens,Hq,Hkv,D", [
    ([1], 1, 1, 64), ([1, 1, 2, 3], 2, 1, 64), ([128], 2, 2, 128), ([129, 255, 257], 4, 2, 128),
    ([700], 2, 1, 128), ([300, 77, 1, 513, 64], 4, 4, 64), ([1100, 5], 8, 2, 128)])
def test_packed_documents(lens, Hq, Hkv, D):
    w = Workload("packed", Hq, Hkv, D, [(L, 1, 0) for L in lens], 77)
    _run(w)


@pytest.mark.parametrize("L,N,r", [(2048, 4, 0), (2048, 4, 1), (2048, 4, 3), (1999, 4, 2),
                                    (50, 4, 1), (7, 4, 0), (3000, 3, 1)])
def test_zigzag_cp_steps_and_merge(L, N, r):
    w = Workload("cp", 4, 2, 128, [(L, N, r)], 91 + r)
    _run(w)


def test_mixed_hdp_buffer():
    w = Workload("mixed", 4, 1, 128, [(50, 4, 1), (7, 1, 0), (1200, 2, 0), (300, 1, 0)], 5)
    _run(w)
