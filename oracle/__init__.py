"""ctypes loader for the fp64 CPU oracle (oracle/sangam_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package never imports this module
and this module never imports the product package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sangam_oracle.c")
_LIB = os.path.join(_HERE, "libsangam_oracle.so")
CFLAGS = ["-O2", "-fopenmp", "-shared", "-fPIC"]
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp the oracle into oracle/libsangam_oracle.so (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", *CFLAGS, "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
    return _lib


def _p(a: np.ndarray, ty):
    return a.ctypes.data_as(ctypes.POINTER(ty))


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def kv_write(k, v, slot_mapping, k_pages, v_pages):
    """In place on k_pages, v_pages (uint16 [P][Hkv][16][D])."""
    k = np.ascontiguousarray(k, np.uint16)
    v = np.ascontiguousarray(v, np.uint16)
    sm = np.ascontiguousarray(slot_mapping, np.int32)
    assert k_pages.flags.c_contiguous and v_pages.flags.c_contiguous
    _, Hkv, _, D = k_pages.shape
    rc = lib().oracle_kv_write(_p(k, ctypes.c_uint16), _p(v, ctypes.c_uint16), _p(sm, ctypes.c_int32),
                               ctypes.c_int32(len(sm)), ctypes.c_int32(Hkv), ctypes.c_int32(D),
                               _p(k_pages, ctypes.c_uint16), _p(v_pages, ctypes.c_uint16))
    assert rc == 0


def block_attn(q, k_pages, v_pages, block_table, cu_q_lens, ctx_lens, scale, rows=None, want_aux=False):
    """fp64 attention output [T_q or len(rows)][Hq][D] (+ lse, rowsum when want_aux)."""
    q = np.ascontiguousarray(q, np.uint16)
    bt = np.ascontiguousarray(block_table, np.int32)
    cu = np.ascontiguousarray(cu_q_lens, np.int32)
    cl = np.ascontiguousarray(ctx_lens, np.int32)
    R = len(cl)
    W = bt.shape[1] if bt.ndim == 2 and bt.shape[0] else 1
    _, Hq, D = q.shape if q.ndim == 3 else (0, q.shape[-2], q.shape[-1])
    Hkv = k_pages.shape[1]
    if rows is not None:
        rows = np.ascontiguousarray(rows, np.int32)
        n = len(rows)
        rp = _p(rows, ctypes.c_int32)
    else:
        n = int(cu[-1])
        rp = ctypes.POINTER(ctypes.c_int32)()
    out = np.zeros((n, Hq, D), np.float64)
    lse = np.zeros((n, Hq), np.float64)
    rs = np.zeros((n, Hq), np.float64)
    rc = lib().oracle_block_attn(
        _p(q, ctypes.c_uint16), _p(k_pages, ctypes.c_uint16), _p(v_pages, ctypes.c_uint16),
        _p(bt, ctypes.c_int32), ctypes.c_int32(W), _p(cu, ctypes.c_int32), _p(cl, ctypes.c_int32),
        ctypes.c_int32(R), ctypes.c_int32(Hq), ctypes.c_int32(Hkv), ctypes.c_int32(D),
        ctypes.c_float(float(np.float32(scale))), rp, ctypes.c_int32(n),
        _p(out, ctypes.c_double),
        _p(lse, ctypes.c_double) if want_aux else ctypes.POINTER(ctypes.c_double)(),
        _p(rs, ctypes.c_double) if want_aux else ctypes.POINTER(ctypes.c_double)())
    assert rc == 0
    return (out, lse, rs) if want_aux else out


def attn_contiguous(q, k, v, cu_ctx, cu_q_lens, scale):
    q = np.ascontiguousarray(q, np.uint16)
    k = np.ascontiguousarray(k, np.uint16)
    v = np.ascontiguousarray(v, np.uint16)
    cc = np.ascontiguousarray(cu_ctx, np.int64)
    cu = np.ascontiguousarray(cu_q_lens, np.int32)
    T, Hq, D = q.shape
    Hkv = k.shape[1]
    out = np.zeros((T, Hq, D), np.float64)
    rc = lib().oracle_attn_contiguous(
        _p(q, ctypes.c_uint16), _p(k, ctypes.c_uint16), _p(v, ctypes.c_uint16),
        _p(cc, ctypes.c_int64), _p(cu, ctypes.c_int32), ctypes.c_int32(len(cu) - 1),
        ctypes.c_int32(Hq), ctypes.c_int32(Hkv), ctypes.c_int32(D),
        ctypes.c_float(float(np.float32(scale))), _p(out, ctypes.c_double))
    assert rc == 0
    return out


def combine(O_parts, m_parts, l_parts):
    O = np.ascontiguousarray(O_parts, np.float64)
    m = np.ascontiguousarray(m_parts, np.float64)
    l = np.ascontiguousarray(l_parts, np.float64)
    n, D = O.shape
    out = np.zeros(D, np.float64)
    rc = lib().oracle_combine(_p(O, ctypes.c_double), _p(m, ctypes.c_double), _p(l, ctypes.c_double),
                              ctypes.c_int32(n), ctypes.c_int32(D), _p(out, ctypes.c_double))
    assert rc == 0
    return out


def iteration(b, rows=None, poison=True):
    """The whole hot path on a sangam_inputs.Batch `b` (duck-typed; no import): load the cache
    content, write this iteration's K/V rows, attend.  Returns (out fp64, k_pages, v_pages)."""
    P, Hkv, D = b.num_pages, b.num_kv_heads, b.head_dim
    fill = np.uint16(0x7FC1) if poison else np.uint16(0)
    kp = np.full((P, Hkv, 16, D), fill, np.uint16)
    vp = np.full((P, Hkv, 16, D), fill, np.uint16)
    kv_write(b.k_cache, b.v_cache, b.slot_cache, kp, vp)
    kv_write(b.k_new, b.v_new, b.slot_new, kp, vp)
    out = block_attn(b.q, kp, vp, b.block_table, b.cu_q_lens, b.ctx_lens, b.scale, rows=rows)
    return out, kp, vp
