"""ctypes loader for the fp64 CPU oracle (oracle/jetlong_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from
paper_2607_07740_b200 and the product never imports it.

All arithmetic lives in the C file; this module only builds it (gcc) and marshals numpy arrays.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "jetlong_oracle.c")
_SO = os.path.join(_HERE, "libjetlong_oracle.so")
_lib = None


def build(force=False):
    """Compile jetlong_oracle.c with gcc (OpenMP, -O2, no fast-math)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-Wall", "-o", _SO, _SRC, "-lm"])
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_SO)
        i64, i32, dbl, vp = ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_void_p
        L.jlo_group_size.restype = i64
        L.jlo_group_size.argtypes = [i64, i64]
        L.jlo_remote_pos.restype = i64
        L.jlo_remote_pos.argtypes = [i64, i64]
        L.jlo_delta.restype = i64
        L.jlo_delta.argtypes = [i64, i64]
        L.jlo_rope.restype = None
        L.jlo_rope.argtypes = [vp, i32, dbl, i64, vp]
        L.jlo_num_threads.restype = i32
        L.jlo_attend_rows.restype = i32
        L.jlo_attend_rows.argtypes = [vp, vp, vp, i64, i32, i32, i32, i64, i64, dbl, i32, i64, i64, vp, vp, vp, vp, vp]
        L.jlo_three_call_rows.restype = i32
        L.jlo_three_call_rows.argtypes = [vp, vp, vp, i64, i32, i32, i32, i64, i64, dbl, i64, vp, vp, vp, vp, vp]
        L.jlo_attend_rows_freq.restype = i32
        L.jlo_attend_rows_freq.argtypes = [vp, vp, vp, i64, i32, i32, i32, i64, i64, dbl, dbl, dbl, i64, i64, vp, vp, vp, vp]
        L.jlo_scores_row.restype = i32
        L.jlo_scores_row.argtypes = [vp, vp, i64, i32, i32, i32, i64, i64, dbl, i32, i64, vp]
        _lib = L
    return _lib


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def group_size(L, w_pre):
    return int(lib().jlo_group_size(int(L), int(w_pre)))


def remote_pos(x, G):
    return int(lib().jlo_remote_pos(int(x), int(G)))


def delta(x, G):
    return int(lib().jlo_delta(int(x), int(G)))


def num_threads():
    return int(lib().jlo_num_threads())


def rope(x, theta, n):
    """RoPE(x, n): rotate pairs (i, i+d/2) of a 1-D float64 vector by n*theta_i."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    y = np.empty_like(x)
    lib().jlo_rope(_p(x), x.shape[0], float(theta), int(n), _p(y))
    return y


def _rows_heads(rows, heads):
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    heads = np.ascontiguousarray(heads, dtype=np.int32)
    assert rows.shape == heads.shape and rows.ndim == 1
    return rows, heads


def attend_rows(Q, K, V, rows, heads, *, w_local, w_pretrained, rope_theta, mode="bifocal", pos_shift=0,
                q_is_compact=False, Ls=None):
    """out[n,d], lse[n] (float64) for the (row, head) pairs.

    Q: [L,H_q,d] (or, with q_is_compact, [n,d] already gathered plus H_q passed via heads max is
    not possible -- so compact callers must pass H_q through Q=(Qrows, H_q)).  K, V: [L,H_kv,d].
    Ls: optional per-pair current length (decode runs): pair j sees keys 0..rows[j] with G from Ls[j].
    """
    K = _f32(K)
    V = _f32(V)
    L, H_kv, d = K.shape
    rows, heads = _rows_heads(rows, heads)
    if q_is_compact:
        Qrows, H_q = Q
        Qrows = _f32(Qrows)
    else:
        H_q = Q.shape[1]
        if rows.size and (rows.min() < 0 or rows.max() >= Q.shape[0] or heads.min() < 0 or heads.max() >= H_q):
            raise ValueError("row/head out of range")
        Qrows = _f32(np.asarray(Q)[rows, heads])
    n = rows.shape[0]
    assert Qrows.shape == (n, d)
    out = np.empty((n, d), dtype=np.float64)
    lse = np.empty((n,), dtype=np.float64)
    if Ls is not None:
        Ls = np.ascontiguousarray(Ls, dtype=np.int64)
        assert Ls.shape == rows.shape
    rc = lib().jlo_attend_rows(_p(Qrows), _p(K), _p(V), L, H_q, H_kv, d, int(w_local), int(w_pretrained),
                               float(rope_theta), {"bifocal": 0, "causal": 1}[mode], int(pos_shift), n,
                               _p(rows), _p(heads), _p(Ls) if Ls is not None else None, _p(out), _p(lse))
    if rc != 0:
        raise ValueError("jlo_attend_rows: bad arguments")
    return out, lse


def attend_rows_freq(Q, K, V, rows, heads, *, w_local, w_pretrained, rope_theta, alpha=1.0, beta=32.0, pos_shift=0,
                     q_is_compact=False):
    """The frequency-interpolation remote map (R17): out[n,d], lse[n] (float64)."""
    K = _f32(K)
    V = _f32(V)
    L, H_kv, d = K.shape
    rows, heads = _rows_heads(rows, heads)
    if q_is_compact:
        Qrows, H_q = Q
        Qrows = _f32(Qrows)
    else:
        H_q = Q.shape[1]
        Qrows = _f32(np.asarray(Q)[rows, heads])
    n = rows.shape[0]
    out = np.empty((n, d), dtype=np.float64)
    lse = np.empty((n,), dtype=np.float64)
    rc = lib().jlo_attend_rows_freq(_p(Qrows), _p(K), _p(V), L, H_q, H_kv, d, int(w_local), int(w_pretrained),
                                    float(rope_theta), float(alpha), float(beta), int(pos_shift), n, _p(rows), _p(heads),
                                    _p(out), _p(lse))
    if rc != 0:
        raise ValueError("jlo_attend_rows_freq: bad arguments")
    return out, lse


def attend_all(Q, K, V, **kw):
    """Every (row, head): out [L,H_q,d], lse [H_q,L]."""
    L, H_q, d = Q.shape
    rows = np.repeat(np.arange(L, dtype=np.int64), H_q)
    heads = np.tile(np.arange(H_q, dtype=np.int32), L)
    out, lse = attend_rows(Q, K, V, rows, heads, **kw)
    return out.reshape(L, H_q, d), lse.reshape(L, H_q).T.copy()


def three_call_rows(Q, K, V, rows, heads, *, w_local, w_pretrained, rope_theta):
    """Literal Section 3.3: calls A, B, C and the Eq.(7) merge.  Returns out, lse, parts[n,3]."""
    K = _f32(K)
    V = _f32(V)
    L, H_kv, d = K.shape
    H_q = Q.shape[1]
    rows, heads = _rows_heads(rows, heads)
    Qrows = _f32(np.asarray(Q)[rows, heads])
    n = rows.shape[0]
    out = np.empty((n, d), dtype=np.float64)
    lse = np.empty((n,), dtype=np.float64)
    parts = np.empty((n, 3), dtype=np.float64)
    rc = lib().jlo_three_call_rows(_p(Qrows), _p(K), _p(V), L, H_q, H_kv, d, int(w_local), int(w_pretrained),
                                   float(rope_theta), n, _p(rows), _p(heads), _p(out), _p(lse), _p(parts))
    if rc != 0:
        raise ValueError("jlo_three_call_rows: bad arguments")
    return out, lse, parts


def scores_row(Qrow, K, q, kv, *, w_local, w_pretrained, rope_theta, mode="bifocal"):
    """Scaled scores s[0..q] of one query row against KV head kv."""
    K = _f32(K)
    L, H_kv, d = K.shape
    Qrow = _f32(Qrow)
    s = np.empty((q + 1,), dtype=np.float64)
    rc = lib().jlo_scores_row(_p(Qrow), _p(K), L, H_kv, int(kv), d, int(w_local), int(w_pretrained),
                              float(rope_theta), {"bifocal": 0, "causal": 1}[mode], int(q), _p(s))
    if rc != 0:
        raise ValueError("jlo_scores_row: bad arguments")
    return s
