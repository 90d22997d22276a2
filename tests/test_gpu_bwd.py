"""-m gpu: forward + merge + backward (prep, bs_attn_bwd per step, finish) through the C-ABI
against the fp64 oracle: every element of dQ, dK, dV on small packed / zigzag-CP workloads."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2502_21231_b200.synth.workloads import Workload  # noqa: E402


def _run(w, fused_clear=False):
    import gpu_util as U
    import oracle
    run = U.DeviceRun(w, fused_clear=fused_clear)
    O, LSE, _ = run.forward()
    U.check_forward(run, O, LSE)
    dQ, grads, _ = run.backward(O, LSE)
    dQo, go = run.oracle_backward()
    got = oracle.bf16_to_f64(U.to_bits(dQ)).reshape(dQo.shape)
    assert not np.isnan(got).any()
    errs = {"dQ": U.rel_l2(got, dQo)}
    gk = np.concatenate([oracle.bf16_to_f64(U.to_bits(grads[s][0])).reshape(go[s][0].shape)
                         for s in run.steps])
    gv = np.concatenate([oracle.bf16_to_f64(U.to_bits(grads[s][1])).reshape(go[s][1].shape)
                         for s in run.steps])
    assert not np.isnan(gk).any() and not np.isnan(gv).any()
    errs["dK"] = U.rel_l2(gk, np.concatenate([go[s][0] for s in run.steps]))
    errs["dV"] = U.rel_l2(gv, np.concatenate([go[s][1] for s in run.steps]))
    for k, v in errs.items():
        assert v <= U.TOL_GRAD, f"{k} relative L2 error {v}"
    return errs


@pytest.mark.parametrize("lens,Hq,Hkv,D", [
    ([1], 1, 1, 64), ([64], 1, 1, 128), ([128], 2, 2, 128), ([129, 255, 257], 4, 2, 128),
    ([700], 2, 1, 128), ([300, 77, 1, 513, 64], 4, 4, 64), ([1100, 5], 8, 2, 128)])
def test_packed_documents(lens, Hq, Hkv, D):
    print(_run(Workload("packed", Hq, Hkv, D, [(L, 1, 0) for L in lens], 78)))


@pytest.mark.parametrize("L,N,r", [(2048, 4, 0), (2048, 4, 1), (2048, 4, 3), (1999, 4, 2),
                                    (50, 4, 1), (3000, 3, 1)])
def test_zigzag_cp(L, N, r):
    print(_run(Workload("cp", 4, 2, 128, [(L, N, r)], 92 + r)))


def test_mixed_hdp_buffer():
    print(_run(Workload("mixed", 4, 1, 128, [(50, 4, 1), (7, 1, 0), (1200, 2, 0), (300, 1, 0)], 6)))


@pytest.mark.parametrize("seqs,Hq,Hkv,D", [
    ([(129, 1, 0), (255, 1, 0), (257, 1, 0)], 4, 2, 128),       # ragged units overhang into the next document
    ([(300, 1, 0), (77, 1, 0), (1, 1, 0), (513, 1, 0)], 4, 4, 64),
    ([(2048, 4, 1)], 4, 2, 128),                                # low part rows see nothing in some steps
    ([(50, 4, 1), (7, 1, 0), (1200, 2, 0), (300, 1, 0)], 4, 1, 128)])
def test_accumulator_cleared_by_forward(seqs, Hq, Hkv, D):
    """dQ_acc (NaN-filled) is cleared by the first step's bs_attn_fwd, prep gets dQ_acc = NULL."""
    print(_run(Workload("fused", Hq, Hkv, D, seqs, 93), fused_clear=True))
