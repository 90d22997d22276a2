"""TEST INFRASTRUCTURE ONLY: ctypes front end of oracle/oracle_attn.c (fp64, plain definition).

See oracle_attn.c for the formulas and the PAPER.md passages they follow.  This file only
marshals numpy arrays; the one piece of arithmetic here is ``bf16_to_f64`` (exact widening).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = os.path.join(_HERE, "oracle_attn.c")
_lib = None


def build(force=False):
    """Compile oracle_attn.c -> liboracle.so with gcc (-O2 -fopenmp).  No fast-math."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11",
                               "-o", _SO, _SRC, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        i64, i32, dbl, vp = ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_void_p
        lib.oracle_threads.restype = ctypes.c_int
        lib.oracle_attn_fwd.restype = ctypes.c_int
        lib.oracle_attn_fwd.argtypes = [i64, i64, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp, dbl,
                                        vp, vp]
        lib.oracle_attn_bwd.restype = ctypes.c_int
        lib.oracle_attn_bwd.argtypes = [i64, i64, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp,
                                        dbl, vp, vp, vp, vp, vp]
        lib.oracle_merge.restype = ctypes.c_int
        lib.oracle_merge.argtypes = [i32, i64, i32, i32, vp, vp, vp, vp]
        _lib = lib
    return _lib


def threads():
    return int(_load().oracle_threads())


def bf16_to_f64(bits):
    """Exact widening of bf16 bit patterns (uint16 array) to float64."""
    bits = np.ascontiguousarray(bits, dtype=np.uint16)
    return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def _u16(a, shape):
    a = np.ascontiguousarray(a, dtype=np.uint16)
    assert a.shape == shape, (a.shape, shape)
    return a


def _i32(a, n):
    a = np.ascontiguousarray(a, dtype=np.int32)
    assert a.shape == (n,), (a.shape, n)
    return a


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def attn_fwd(Q, K, V, q_seq, q_pos, k_seq, k_pos, scale=None):
    """Masked causal softmax attention.  Q [nq,Hq,D], K,V [nk,Hkv,D] bf16 bits (uint16);
    q_seq,q_pos [nq], k_seq,k_pos [nk] int32.  Returns O [nq,Hq,D] f64, LSE [Hq,nq] f64."""
    nq, Hq, D = Q.shape
    nk, Hkv, _ = K.shape
    scale = float(scale) if scale else 1.0 / np.sqrt(D)
    Q, K, V = _u16(Q, (nq, Hq, D)), _u16(K, (nk, Hkv, D)), _u16(V, (nk, Hkv, D))
    q_seq, q_pos, k_seq, k_pos = _i32(q_seq, nq), _i32(q_pos, nq), _i32(k_seq, nk), _i32(k_pos, nk)
    O = np.empty((nq, Hq, D), np.float64)
    LSE = np.empty((Hq, nq), np.float64)
    rc = _load().oracle_attn_fwd(nq, nk, Hq, Hkv, D, _p(Q), _p(K), _p(V), _p(q_seq), _p(q_pos),
                                 _p(k_seq), _p(k_pos), scale, _p(O), _p(LSE))
    assert rc == 0
    return O, LSE


def attn_bwd(Q, K, V, dO, q_seq, q_pos, k_seq, k_pos, scale=None, LSE=None, delta=None):
    """Gradients of sum(O * dO).  Returns dQ [nq,Hq,D], dK, dV [nk,Hkv,D] f64.
    LSE/delta ([Hq,nq] f64) given => partial gradients w.r.t. this key set under the merged
    normaliser; None => the plain definition over this key set."""
    nq, Hq, D = Q.shape
    nk, Hkv, _ = K.shape
    scale = float(scale) if scale else 1.0 / np.sqrt(D)
    Q, K, V = _u16(Q, (nq, Hq, D)), _u16(K, (nk, Hkv, D)), _u16(V, (nk, Hkv, D))
    dO = _u16(dO, (nq, Hq, D))
    q_seq, q_pos, k_seq, k_pos = _i32(q_seq, nq), _i32(q_pos, nq), _i32(k_seq, nk), _i32(k_pos, nk)
    assert (LSE is None) == (delta is None)
    if LSE is not None:
        LSE = np.ascontiguousarray(LSE, np.float64)
        delta = np.ascontiguousarray(delta, np.float64)
        assert LSE.shape == (Hq, nq) and delta.shape == (Hq, nq)
    dQ = np.empty((nq, Hq, D), np.float64)
    dK = np.empty((nk, Hkv, D), np.float64)
    dV = np.empty((nk, Hkv, D), np.float64)
    rc = _load().oracle_attn_bwd(nq, nk, Hq, Hkv, D, _p(Q), _p(K), _p(V), _p(dO), _p(q_seq),
                                 _p(q_pos), _p(k_seq), _p(k_pos), scale,
                                 _p(LSE) if LSE is not None else None,
                                 _p(delta) if delta is not None else None, _p(dQ), _p(dK), _p(dV))
    assert rc == 0
    return dQ, dK, dV


def merge(O_parts, LSE_parts):
    """O_parts [n,rows,Hq,D] f64, LSE_parts [n,Hq,rows] f64 -> O [rows,Hq,D], LSE [Hq,rows]."""
    O_parts = np.ascontiguousarray(O_parts, np.float64)
    LSE_parts = np.ascontiguousarray(LSE_parts, np.float64)
    n, rows, Hq, D = O_parts.shape
    assert LSE_parts.shape == (n, Hq, rows)
    O = np.empty((rows, Hq, D), np.float64)
    LSE = np.empty((Hq, rows), np.float64)
    rc = _load().oracle_merge(n, rows, Hq, D, _p(O_parts), _p(LSE_parts), _p(O), _p(LSE))
    assert rc == 0
    return O, LSE


def rows_from_plan(pl, step=None):
    """(seq, pos) int32 arrays of the local Q rows (step None) or of step `step`'s KV rows of an
    oracle plan (oracle/plan.py) — the global positions the mask is defined on."""
    if step is None:
        return pl["q_seq"].copy(), pl["q_pos"].copy()
    st = pl["steps"][step]
    return st["k_seq"].copy(), st["k_pos"].copy()
