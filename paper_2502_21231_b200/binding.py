"""Thin ctypes binding of csrc/libbytescale_attn.so — same names as include/bytescale_attn.h.

Argument marshalling only: every step of the path runs in the library's kernels.  PyTorch
appears here only as the owner of device memory (``tensor.data_ptr()``) and of the stream.
Fails loudly (ImportError) when the shared library has not been built: there is no fallback.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libbytescale_attn.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2502_21231_b200.build` "
                      "(there is no CPU or PyTorch fallback)")
lib = ctypes.CDLL(LIB_PATH)

BS_OK = 0
BS_MAX_MERGE_PARTS = 64


class BsError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__(f"{where}: {lib.bs_status_string(code).decode()} — "
                         f"{lib.bs_last_error().decode()}")


class Seq(ctypes.Structure):
    _fields_ = [("len", ctypes.c_int32), ("cp", ctypes.c_int32), ("rank", ctypes.c_int32)]


class Seg(ctypes.Structure):
    _fields_ = [("q_begin", ctypes.c_int32), ("q_end", ctypes.c_int32), ("k_begin", ctypes.c_int32),
                ("k_end", ctypes.c_int32), ("causal_offset", ctypes.c_int32), ("seq", ctypes.c_int32)]


class Step(ctypes.Structure):
    _fields_ = [("step", ctypes.c_int32), ("n_segs", ctypes.c_int32),
                ("segs", ctypes.POINTER(Seg)), ("kv_rows", ctypes.c_int32),
                ("n_kv_seqs", ctypes.c_int32), ("kv_seq", ctypes.POINTER(ctypes.c_int32)),
                ("kv_src_rank", ctypes.POINTER(ctypes.c_int32)),
                ("cu_rows_k", ctypes.POINTER(ctypes.c_int32)), ("visible_pairs", ctypes.c_int64)]


class Shape(ctypes.Structure):
    _fields_ = [("n_q_heads", ctypes.c_int32), ("n_kv_heads", ctypes.c_int32),
                ("head_dim", ctypes.c_int32), ("softmax_scale", ctypes.c_float),
                ("q_rows", ctypes.c_int32), ("kv_rows", ctypes.c_int32),
                ("q_row_stride", ctypes.c_int64), ("kv_row_stride", ctypes.c_int64),
                ("lse_head_stride", ctypes.c_int64)]


_vp, _i32, _i64, _sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_size_t
_P = ctypes.POINTER
lib.bs_status_string.restype = ctypes.c_char_p
lib.bs_status_string.argtypes = [ctypes.c_int]
lib.bs_last_error.restype = ctypes.c_char_p
lib.bs_version.restype = ctypes.c_int
lib.bs_plan.argtypes = [_P(Seq), _i32, _P(_vp)]
lib.bs_plan_uniform.argtypes = [_P(_i32), _i32, _i32, _i32, _i32, _P(_vp)]
for _n in ("bs_plan_n_seqs", "bs_plan_q_rows", "bs_plan_n_steps"):
    getattr(lib, _n).restype = _i32
    getattr(lib, _n).argtypes = [_vp]
for _n in ("bs_plan_cu_rows_q", "bs_plan_q_pos", "bs_plan_q_seq"):
    getattr(lib, _n).restype = _P(_i32)
    getattr(lib, _n).argtypes = [_vp]
for _n in ("bs_plan_step_k_pos", "bs_plan_step_k_seq"):
    getattr(lib, _n).restype = _P(_i32)
    getattr(lib, _n).argtypes = [_vp, _i32]
lib.bs_plan_step.restype = _P(Step)
lib.bs_plan_step.argtypes = [_vp, _i32]
lib.bs_plan_destroy.restype = None
lib.bs_plan_destroy.argtypes = [_vp]


class Microbatch(ctypes.Structure):
    _fields_ = [("round", _i32), ("rank", _i32), ("n_seqs", _i32), ("seqs", _P(Seq)),
                ("src", _P(_i32))]


lib.bs_assign.argtypes = [_P(_i32), _i32, _i32, _i32, _P(_vp)]
for _n in ("bs_assign_n_rounds", "bs_assign_n_seqs", "bs_assign_n_microbatches"):
    getattr(lib, _n).restype = _i32
    getattr(lib, _n).argtypes = [_vp]
lib.bs_assign_ranks_needed.restype = _P(_i32)
lib.bs_assign_ranks_needed.argtypes = [_vp]
lib.bs_assign_microbatch.restype = _P(Microbatch)
lib.bs_assign_microbatch.argtypes = [_vp, _i32]
lib.bs_assign_destroy.restype = None
lib.bs_assign_destroy.argtypes = [_vp]


class TimedMicrobatch(ctypes.Structure):
    _fields_ = [("rank", _i32), ("n_seqs", _i32), ("start", _i64), ("end", _i64),
                ("seqs", _P(Seq)), ("src", _P(_i32))]


lib.bs_balance.argtypes = [_P(_i32), _i32, _i32, _i32, _P(_i64), _i32, _i64, _P(_vp)]
for _n in ("bs_balance_n_ranks", "bs_balance_n_microbatches"):
    getattr(lib, _n).restype = _i32
    getattr(lib, _n).argtypes = [_vp]
lib.bs_balance_exec_times.restype = _P(_i64)
lib.bs_balance_exec_times.argtypes = [_vp]
lib.bs_balance_makespan.restype = _i64
lib.bs_balance_makespan.argtypes = [_vp]
lib.bs_balance_microbatch.restype = _P(TimedMicrobatch)
lib.bs_balance_microbatch.argtypes = [_vp, _i32]
lib.bs_balance_destroy.restype = None
lib.bs_balance_destroy.argtypes = [_vp]
lib.bs_attn_workspace_bytes.argtypes = [_P(Shape), _i32, ctypes.c_int, _P(_sz)]
lib.bs_attn_fwd.argtypes = [_P(Shape), _vp, _vp, _vp, _P(Seg), _i32, _i32, _i32, _vp, _vp, _vp,
                            _sz, _vp, _vp]
lib.bs_attn_fwd_static.argtypes = [_P(Shape), _vp, _vp, _vp, _P(Seg), _i32, _i32, _i32, _vp, _vp,
                                   _vp, _vp]
lib.bs_attn_bwd_prep.argtypes = [_P(Shape), _vp, _vp, _vp, _vp, _vp]
lib.bs_attn_bwd.argtypes = [_P(Shape), _vp, _vp, _vp, _vp, _vp, _vp, _P(Seg), _i32, _vp, _vp, _vp,
                            _vp, _sz, _vp]
lib.bs_attn_bwd_finish.argtypes = [_P(Shape), _vp, _vp, _vp]
lib.bs_lse_merge.argtypes = [_i32, _P(_vp), _P(_vp), _P(Shape), _i32, _i32, _vp, _vp, _vp]
lib.bs_softmax_xent.argtypes = [_vp, _vp, _i32, _i32, _i64, ctypes.c_float, _vp, _vp, _vp]
lib.bs_hbm_probe.argtypes = [_i32, _P(_vp), _vp, _vp, _sz, _vp]
lib.bs_reduce_probe.argtypes = [_vp, _i32, _i32, _i32, _i32, _vp]
lib.bs_launch_count.restype = _i64
lib.bs_launch_count_reset.restype = None

EXPORTS = ["bs_status_string", "bs_last_error", "bs_version", "bs_plan", "bs_plan_uniform",
           "bs_plan_n_seqs", "bs_plan_q_rows", "bs_plan_cu_rows_q", "bs_plan_q_pos",
           "bs_plan_q_seq", "bs_plan_n_steps", "bs_plan_step", "bs_plan_step_k_pos",
           "bs_plan_step_k_seq", "bs_plan_destroy", "bs_assign", "bs_assign_n_rounds",
           "bs_assign_n_seqs", "bs_assign_ranks_needed", "bs_assign_n_microbatches",
           "bs_assign_microbatch", "bs_assign_destroy", "bs_balance", "bs_balance_n_ranks",
           "bs_balance_exec_times", "bs_balance_makespan", "bs_balance_n_microbatches",
           "bs_balance_microbatch", "bs_balance_destroy", "bs_attn_workspace_bytes", "bs_attn_fwd",
           "bs_attn_bwd_prep", "bs_attn_bwd", "bs_attn_bwd_finish", "bs_lse_merge", "bs_softmax_xent",
           "bs_hbm_probe", "bs_attn_fwd_static", "bs_reduce_probe",
           "bs_launch_count", "bs_launch_count_reset"]


def _check(code, where):
    if code != BS_OK:
        raise BsError(code, where)


def _arr(ptr, n):
    return np.ctypeslib.as_array(ptr, shape=(n,)).copy() if n > 0 else np.zeros(0, np.int32)


def _plan_to_dict(h):
    n_seqs, q_rows, n_steps = lib.bs_plan_n_seqs(h), lib.bs_plan_q_rows(h), lib.bs_plan_n_steps(h)
    steps = []
    for s in range(n_steps):
        st = lib.bs_plan_step(h, s).contents
        segs = [(g.q_begin, g.q_end, g.k_begin, g.k_end, g.causal_offset, g.seq)
                for g in (st.segs[i] for i in range(st.n_segs))]
        steps.append(dict(step=st.step, segs=segs, kv_rows=st.kv_rows,
                          kv_seq=_arr(st.kv_seq, st.n_kv_seqs).tolist(),
                          kv_src_rank=_arr(st.kv_src_rank, st.n_kv_seqs).tolist(),
                          cu_rows_k=_arr(st.cu_rows_k, st.n_kv_seqs + 1).tolist(),
                          visible_pairs=int(st.visible_pairs),
                          k_pos=_arr(lib.bs_plan_step_k_pos(h, s), st.kv_rows),
                          k_seq=_arr(lib.bs_plan_step_k_seq(h, s), st.kv_rows)))
    return dict(n_seqs=n_seqs, q_rows=q_rows, cu_rows_q=_arr(lib.bs_plan_cu_rows_q(h), n_seqs + 1).tolist(),
                q_pos=_arr(lib.bs_plan_q_pos(h), q_rows), q_seq=_arr(lib.bs_plan_q_seq(h), q_rows),
                n_steps=n_steps, steps=steps)


def plan(seqs):
    """bs_plan: [(len, cp, rank), ...] -> dict copy of the plan (same keys as the C accessors)."""
    seqs = list(seqs)
    arr = (Seq * max(len(seqs), 1))(*[Seq(*map(int, s)) for s in seqs])
    h = _vp()
    _check(lib.bs_plan(arr, len(seqs), ctypes.byref(h)), "bs_plan")
    try:
        return _plan_to_dict(h)
    finally:
        lib.bs_plan_destroy(h)


def assign(lens, capacity, d_hdp):
    """bs_assign: global batch of lengths -> {"d": [D(s_i)], "n_rounds": R, "microbatches":
    [(round, rank, [(len, cp, cp_rank, input index), ...]), ...]} in (round, rank) order."""
    lens = [int(x) for x in lens]
    arr = (_i32 * max(len(lens), 1))(*lens)
    h = _vp()
    _check(lib.bs_assign(arr, len(lens), int(capacity), int(d_hdp), ctypes.byref(h)), "bs_assign")
    try:
        n = lib.bs_assign_n_seqs(h)
        d = lib.bs_assign_ranks_needed(h)
        mbs = []
        for k in range(lib.bs_assign_n_microbatches(h)):
            m = lib.bs_assign_microbatch(h, k).contents
            mbs.append((m.round, m.rank, [(m.seqs[i].len, m.seqs[i].cp, m.seqs[i].rank, m.src[i])
                                          for i in range(m.n_seqs)]))
        return {"d": [d[i] for i in range(n)], "n_rounds": lib.bs_assign_n_rounds(h),
                "microbatches": mbs}
    finally:
        lib.bs_assign_destroy(h)


def balance(lens, capacity, d_hdp, cost, n_buckets=4, delta=0):
    """bs_balance: {"exec_times": [d_hdp], "makespan", "microbatches": [(rank, start, end,
    [(len, cp, cp_rank, input index), ...]), ...]} in (rank, start) order."""
    lens = [int(x) for x in lens]
    arr = (_i32 * max(len(lens), 1))(*lens)
    c = (_i64 * 3)(*[int(x) for x in cost])
    h = _vp()
    _check(lib.bs_balance(arr, len(lens), int(capacity), int(d_hdp), c, int(n_buckets), int(delta),
                          ctypes.byref(h)), "bs_balance")
    try:
        t = lib.bs_balance_exec_times(h)
        mbs = []
        for k in range(lib.bs_balance_n_microbatches(h)):
            m = lib.bs_balance_microbatch(h, k).contents
            mbs.append((m.rank, m.start, m.end,
                        [(m.seqs[i].len, m.seqs[i].cp, m.seqs[i].rank, m.src[i]) for i in range(m.n_seqs)]))
        return {"exec_times": [t[i] for i in range(lib.bs_balance_n_ranks(h))],
                "makespan": lib.bs_balance_makespan(h), "microbatches": mbs}
    finally:
        lib.bs_balance_destroy(h)


def plan_uniform(lens, cp, rank, min_shard_len):
    lens = [int(x) for x in lens]
    arr = (_i32 * max(len(lens), 1))(*lens)
    h = _vp()
    _check(lib.bs_plan_uniform(arr, len(lens), cp, rank, min_shard_len, ctypes.byref(h)),
           "bs_plan_uniform")
    try:
        return _plan_to_dict(h)
    finally:
        lib.bs_plan_destroy(h)


def make_shape(n_q_heads, n_kv_heads, head_dim, q_rows, kv_rows, softmax_scale=0.0,
               q_row_stride=None, kv_row_stride=None, lse_head_stride=None):
    return Shape(n_q_heads, n_kv_heads, head_dim, softmax_scale, q_rows, kv_rows,
                 q_row_stride or n_q_heads * head_dim, kv_row_stride or n_kv_heads * head_dim,
                 lse_head_stride or q_rows)


def make_segs(segs):
    segs = list(segs)
    return (Seg * max(len(segs), 1))(*[Seg(*map(int, s)) for s in segs]), len(segs)


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream():
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def attn_workspace_bytes(shape, n_segs, bwd):
    out = _sz()
    _check(lib.bs_attn_workspace_bytes(ctypes.byref(shape), n_segs, int(bool(bwd)),
                                       ctypes.byref(out)), "bs_attn_workspace_bytes")
    return int(out.value)


def attn_fwd(shape, Q, K, V, segs, out_rows, O, LSE, ws, dQ_acc_clear=None):
    sarr, n = make_segs(segs)
    _check(lib.bs_attn_fwd(ctypes.byref(shape), _ptr(Q), _ptr(K), _ptr(V), sarr, n, out_rows[0],
                           out_rows[1], _ptr(O), _ptr(LSE), _ptr(ws), ws.numel() * ws.element_size(),
                           _stream(), None if dQ_acc_clear is None else _ptr(dQ_acc_clear)),
           "bs_attn_fwd")


STATIC_SCRATCH_BYTES = 262144  # BS_ATTN_STATIC_SCRATCH_BYTES


def attn_fwd_static(shape, Q, K, V, segs, out_rows, O, LSE, dQ_acc_clear=None):
    """bs_attn_fwd_static: bs_attn_fwd without a caller workspace (library-owned static scratch)."""
    sarr, n = make_segs(segs)
    _check(lib.bs_attn_fwd_static(ctypes.byref(shape), _ptr(Q), _ptr(K), _ptr(V), sarr, n,
                                  out_rows[0], out_rows[1], _ptr(O), _ptr(LSE), _stream(),
                                  None if dQ_acc_clear is None else _ptr(dQ_acc_clear)),
           "bs_attn_fwd_static")


def attn_bwd_prep(shape, O_final, dO, delta, dQ_acc):
    _check(lib.bs_attn_bwd_prep(ctypes.byref(shape), _ptr(O_final), _ptr(dO), _ptr(delta),
                                None if dQ_acc is None else _ptr(dQ_acc), _stream()),
           "bs_attn_bwd_prep")


def attn_bwd(shape, Q, K, V, dO, LSE_final, delta, segs, dQ_acc, dK, dV, ws):
    sarr, n = make_segs(segs)
    _check(lib.bs_attn_bwd(ctypes.byref(shape), _ptr(Q), _ptr(K), _ptr(V), _ptr(dO), _ptr(LSE_final),
                           _ptr(delta), sarr, n, _ptr(dQ_acc), _ptr(dK), _ptr(dV), _ptr(ws),
                           ws.numel() * ws.element_size(), _stream()), "bs_attn_bwd")


def attn_bwd_finish(shape, dQ_acc, dQ):
    _check(lib.bs_attn_bwd_finish(ctypes.byref(shape), _ptr(dQ_acc), _ptr(dQ), _stream()),
           "bs_attn_bwd_finish")


def lse_merge(O_parts, LSE_parts, shape, rows, O_out, LSE_out):
    n = len(O_parts)
    op = (_vp * n)(*[t.data_ptr() for t in O_parts])
    lp = (_vp * n)(*[t.data_ptr() for t in LSE_parts])
    _check(lib.bs_lse_merge(n, op, lp, ctypes.byref(shape), rows[0], rows[1], _ptr(O_out),
                            _ptr(LSE_out), _stream()), "bs_lse_merge")


def softmax_xent(logits, labels, grad_scale, loss, dlogits, vocab=None):
    """bs_softmax_xent on torch device tensors: logits / dlogits bf16 [T, row_stride], labels
    int32 [T], loss fp32 [T]; vocab defaults to the row width."""
    T, stride = logits.shape
    _check(lib.bs_softmax_xent(_ptr(logits), _ptr(labels), T, stride if vocab is None else vocab,
                               stride, float(grad_scale), _ptr(loss), _ptr(dlogits), _stream()),
           "bs_softmax_xent")


def hbm_probe(ins, out, sink):
    """bs_hbm_probe on torch device tensors: ins = list of equally sized tensors, out = tensor of
    that size or None (pure read), sink = a 4-byte device tensor."""
    n = len(ins)
    arr = (_vp * n)(*[t.data_ptr() for t in ins])
    _check(lib.bs_hbm_probe(n, arr, _ptr(out), _ptr(sink), ins[0].numel() * ins[0].element_size(),
                            _stream()), "bs_hbm_probe")


def reduce_probe(acc, boxes_per_cta):
    """bs_reduce_probe on a torch device tensor acc fp32 [rows][heads][head_dim] (left unchanged)."""
    rows, heads, hd = acc.shape
    _check(lib.bs_reduce_probe(_ptr(acc), rows, heads, hd, boxes_per_cta, _stream()), "bs_reduce_probe")


def launch_count():
    return int(lib.bs_launch_count())


def launch_count_reset():
    lib.bs_launch_count_reset()
