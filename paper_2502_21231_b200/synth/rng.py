"""ctypes front end of synth.c (counter-based SplitMix64 + Box-Muller -> bf16 bits)."""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libsynth.so")
_SRC = os.path.join(_HERE, "synth.c")
_lib = None

STREAM_LENGTHS, STREAM_Q, STREAM_K, STREAM_V, STREAM_DO = 0, 1, 2, 3, 4


def build(force=False):
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11",
                               "-o", _SO, _SRC, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        u64, vp = ctypes.c_uint64, ctypes.c_void_p
        for f in (lib.synth_uniform_f64, lib.synth_normal_f64):
            f.restype = None
            f.argtypes = [u64, u64, u64, u64, u64, vp]
        lib.synth_rows_bf16.restype = None
        lib.synth_rows_bf16.argtypes = [u64, u64, u64, u64, u64, u64, vp]
        _lib = lib
    return _lib


def uniform_f64(seed, stream, seq, start, count):
    out = np.empty(count, np.float64)
    _load().synth_uniform_f64(seed, stream, seq, start, count, out.ctypes.data_as(ctypes.c_void_p))
    return out


def normal_f64(seed, stream, seq, start, count):
    out = np.empty(count, np.float64)
    _load().synth_normal_f64(seed, stream, seq, start, count, out.ctypes.data_as(ctypes.c_void_p))
    return out


def rows_bf16(seed, stream, seq, pos_begin, n_rows, row_elems, out=None):
    """bf16 bit patterns (uint16) of rows [pos_begin, pos_begin+n_rows) of the N(0,1) tensor of
    (seed, stream, seq); shape [n_rows, row_elems].  `out` may be a preallocated uint16 view."""
    if out is None:
        out = np.empty((n_rows, row_elems), np.uint16)
    assert out.dtype == np.uint16 and out.size == n_rows * row_elems and out.flags.c_contiguous
    _load().synth_rows_bf16(seed, stream, seq, pos_begin, n_rows, row_elems,
                            out.ctypes.data_as(ctypes.c_void_p))
    return out
