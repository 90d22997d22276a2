"""-m gpu, collected last on purpose (a failure here hides no other test under `pytest -x`):
bs_attn_fwd_static, the forward for callers that may not allocate device memory (scratch in a
static __device__ array of BS_ATTN_STATIC_SCRATCH_BYTES inside the library, see
include/bytescale_attn.h), against the existing path bs_attn_fwd with a caller workspace.

Both run the same kernels on the same work list, and a unit's arithmetic does not depend on which
CTA pulls it, so O, LSE and the cleared accumulator must agree BIT FOR BIT - tighter than the
tolerance of the oracle comparisons (tests/gpu_util.py), which the existing path is held to by
test_gpu_fwd.py / test_gpu_bwd.py.  Every comparison is made on two calls in a row on one
stream with no synchronisation in between and different work lists (the second one shorter, so
the tail of the first call's tables is still in the array), then once more in the first shape.
"""
import pytest
import torch

pytestmark = pytest.mark.gpu

from paper_2502_21231_b200 import binding as B  # noqa: E402
from paper_2502_21231_b200.synth.workloads import Workload  # noqa: E402


def _nan(shape, dtype):
    return torch.full(shape, float("nan"), dtype=dtype, device="cuda")


class _Case:
    """Inputs of every ring step of one workload on the device, outputs of both paths."""

    def __init__(self, w, clear_acc):
        import gpu_util as U
        self.run = run = U.DeviceRun(w)
        self.clear_acc = clear_acc
        self.Q = U.to_dev(run.Q_bits)
        self.KV = {s: (U.to_dev(run.K_bits[s]), U.to_dev(run.V_bits[s])) for s in run.steps}
        self.ws = {s: torch.empty(B.attn_workspace_bytes(run.shape(s), len(run.plan["steps"][s]["segs"]),
                                                         False), dtype=torch.uint8, device="cuda")
                   for s in run.steps}
        self.out = {}
        for tag in ("ref", "static"):
            self.out[tag] = {s: (_nan((run.q_rows, run.Hq, run.D), torch.bfloat16),
                                 _nan((run.Hq, run.q_rows), torch.float32),
                                 _nan((run.q_rows, run.Hq, run.D), torch.float32) if clear_acc else None)
                             for s in run.steps}

    def reset(self, tag):
        for O, LSE, acc in self.out[tag].values():
            O.fill_(float("nan"))
            LSE.fill_(float("nan"))
            if acc is not None:
                acc.fill_(float("nan"))

    def launch(self, tag):
        run = self.run
        for s in run.steps:
            K, V = self.KV[s]
            O, LSE, acc = self.out[tag][s]
            segs = run.plan["steps"][s]["segs"]
            if tag == "ref":
                B.attn_fwd(run.shape(s), self.Q, K, V, segs, (0, run.q_rows), O, LSE, self.ws[s], acc)
            else:
                B.attn_fwd_static(run.shape(s), self.Q, K, V, segs, (0, run.q_rows), O, LSE, acc)

    def compare(self, label):
        for s in self.run.steps:
            for name, a, b in zip(("O", "LSE", "dQ_acc"), self.out["static"][s], self.out["ref"][s]):
                if a is None:
                    continue
                ia = a.view(torch.int16 if a.dtype == torch.bfloat16 else torch.int32)
                ib = b.view(torch.int16 if b.dtype == torch.bfloat16 else torch.int32)
                n_diff = int((ia != ib).sum())
                assert n_diff == 0, f"{label} step {s}: {name} differs in {n_diff} elements"
                assert not bool(torch.isnan(b.float()).any()), f"{label} step {s}: {name} has NaN"


def _cases():
    # A: a mixed HDP buffer (zigzag shards next to whole documents, ragged ends: clipped tensor
    #    maps, uncovered-row fill in the later ring steps, several launches of table chunks)
    a = Workload("static_a", 8, 2, 128, [(50, 4, 1), (7, 1, 0), (1200, 2, 0), (300, 1, 0), (1, 1, 0),
                                         (2049, 4, 3), (129, 1, 0)] + [(37 + 5 * i, 1, 0) for i in range(40)],
                 501)
    # B: other heads / head dim and a much shorter work list
    b = Workload("static_b", 6, 3, 64, [(257, 1, 0), (100, 2, 1)], 502)
    return _Case(a, clear_acc=True), _Case(b, clear_acc=False)


def test_static_scratch_forward_matches_workspace_forward_twice_in_a_row():
    ca, cb = _cases()
    for c in (ca, cb):          # existing path first
        c.launch("ref")
    torch.cuda.synchronize()
    for rnd in range(2):
        for c in (ca, cb, ca):  # back to back on one stream, nothing in between
            c.launch("static")
            # (the outputs of the first launch of `ca` are overwritten by the third, same values)
        torch.cuda.synchronize()
        ca.compare(f"round {rnd}, A")
        cb.compare(f"round {rnd}, B")
        for c in (ca, cb):
            c.reset("static")
        torch.cuda.synchronize()


def test_static_scratch_forward_allocates_no_device_memory():
    ca, cb = _cases()
    for c in (ca, cb):
        c.launch("ref")
        c.launch("static")      # first use: module load, cudaGetSymbolAddress, kernel attributes
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        ca.launch("static")
        cb.launch("static")
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, f"device memory in use grew by {free0 - free1} bytes"
    ca.compare("A")
    cb.compare("B")


def test_static_scratch_rejects_work_lists_beyond_its_size():
    # 20000 one-row documents: 20000 items, spans, groups and clipped tensor maps, ~3.9 MB of
    # tables against the 256 KiB array
    n, Hq, Hkv, D = 20000, 2, 1, 64
    sh = B.make_shape(Hq, Hkv, D, n, n)
    assert B.attn_workspace_bytes(sh, n, False) > B.STATIC_SCRATCH_BYTES
    Q = torch.zeros((n, Hq, D), dtype=torch.bfloat16, device="cuda")
    K = torch.zeros((n, Hkv, D), dtype=torch.bfloat16, device="cuda")
    O = _nan((n, Hq, D), torch.bfloat16)
    LSE = _nan((Hq, n), torch.float32)
    segs = [(i, i + 1, i, i + 1, 0, i) for i in range(n)]
    with pytest.raises(B.BsError) as e:
        B.attn_fwd_static(sh, Q, K, K, segs, (0, n), O, LSE)
    assert e.value.code == -3, str(e.value)                      # BS_ERR_WORKSPACE
    assert str(B.STATIC_SCRATCH_BYTES) in str(e.value) and "bs_attn_fwd" in str(e.value), str(e.value)
    torch.cuda.synchronize()
    assert bool(torch.isnan(O.float()).all()) and bool(torch.isnan(LSE).all())   # nothing enqueued
    # the existing path takes the same call
    ws = torch.empty(B.attn_workspace_bytes(sh, n, False), dtype=torch.uint8, device="cuda")
    B.attn_fwd(sh, Q, K, K, segs, (0, n), O, LSE, ws)
    torch.cuda.synchronize()
    assert not bool(torch.isnan(O.float()).any())
    # and a call that fits still works afterwards: one key per row, q = k = v = 0, so O = 0 and
    # LSE = ln 1 up to the kernel's exp2 / log approximations, and bit-equal to the existing path
    small = segs[:100]
    sh2 = B.make_shape(Hq, Hkv, D, 100, 100)
    O2, L2 = _nan((100, Hq, D), torch.bfloat16), _nan((Hq, 100), torch.float32)
    O3, L3 = _nan((100, Hq, D), torch.bfloat16), _nan((Hq, 100), torch.float32)
    B.attn_fwd_static(sh2, Q[:100], K[:100], K[:100], small, (0, 100), O2, L2)
    B.attn_fwd(sh2, Q[:100], K[:100], K[:100], small, (0, 100), O3, L3, ws)
    torch.cuda.synchronize()
    assert bool((O2.float() == 0).all()) and float(L2.abs().max()) < 1e-3
    assert torch.equal(O2.view(torch.int16), O3.view(torch.int16))
    assert torch.equal(L2.view(torch.int32), L3.view(torch.int32))


def test_static_scratch_forward_replays_from_a_cuda_graph():
    """The call enqueues kernels whose inputs travel as kernel parameters (tables included) and
    allocates nothing, so a captured launch can be replayed: capture one call of every ring step
    (after a plain warm-up call: first use sets kernel attributes and resolves the scratch
    address), clear the outputs, replay twice, compare with the existing path."""
    ca, _ = _cases()
    ca.launch("ref")
    ca.launch("static")
    torch.cuda.synchronize()
    ca.reset("static")
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        ca.launch("static")
    torch.cuda.synchronize()
    for rnd in range(2):
        ca.reset("static")
        graph.replay()
        torch.cuda.synchronize()
        ca.compare(f"graph replay {rnd}, A")
