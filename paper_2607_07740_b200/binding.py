"""Thin ctypes binding of libjetlong (include/jetlong.h): argument marshalling only.

Every step of the hot path runs inside the CUDA library.  torch is used for device memory and
streams.  There is no CPU fallback: if libjetlong.so is missing or the device is not a B200-class
GPU, the calls raise.
"""
import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libjetlong.so")
_lib = None

OK, INVALID_ARG, UNSUPPORTED, CUDA_ERROR = 0, 1, 2, 3
BF16, FP32 = 0, 1
OP_PREFILL, OP_DECODE, OP_CAUSAL_PREFILL, OP_CAUSAL_DECODE, OP_PREFILL_PREROTATED, OP_PREFILL_UNFUSED = \
    0, 1, 2, 3, 4, 5
PRECISION_COMPENSATED, PRECISION_FAST, PRECISION_COMPENSATED_F16, PRECISION_COMPENSATED_E5M2 = 0, 1, 2, 3

EXPORTS = ["jetlong_group_size", "jetlong_workspace_bytes", "jetlong_prefill", "jetlong_decode",
           "jetlong_causal_prefill", "jetlong_causal_decode", "jetlong_prefill_host", "jetlong_status_string",
           "jetlong_launch_count", "jetlong_set_prefill_impl", "jetlong_prefill_uses_umma",
           "jetlong_set_prefill_precision", "jetlong_prefill_prerotated", "jetlong_prefill_unfused",
           "jetlong_prefill_opt", "jetlong_prefill_prerotated_opt", "jetlong_host_release", "jetlong_decode_opt",
           "jetlong_decode_paged", "jetlong_decode_paged_workspace_bytes", "jetlong_decode_static",
           "jetlong_decode_static_init"]
DEFAULT = -2                                              # JETLONG_DEFAULT: take the calling thread's default


class Options(ctypes.Structure):
    """jetlong_options (include/jetlong.h): per-call precision / implementation."""
    _fields_ = [("struct_bytes", ctypes.c_uint32), ("precision", ctypes.c_int), ("prefill_impl", ctypes.c_int),
                ("remote_map", ctypes.c_int), ("yarn_alpha", ctypes.c_double), ("yarn_beta", ctypes.c_double)]


MAP_ALIAS, MAP_FREQ_INTERP = 0, 1


def _options(precision=None, impl=None, remote_map=None, yarn=None):
    if precision is None and impl is None and remote_map is None and yarn is None:
        return None
    a, b = (0.0, 0.0) if yarn is None else (float(yarn[0]), float(yarn[1]))
    o = Options(ctypes.sizeof(Options), DEFAULT if precision is None else int(precision), DEFAULT if impl is None else int(impl),
                DEFAULT if remote_map is None else int(remote_map), a, b)
    return ctypes.byref(o)


class JetlongError(RuntimeError):
    def __init__(self, status, text):
        super().__init__("libjetlong status %d: %s" % (status, text))
        self.status = status


def lib():
    """Load libjetlong.so (built in-tree by build.py).  Fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise ImportError("libjetlong.so not built: run `python -m paper_2607_07740_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(_SO)
        i64, i32, dbl, vp, sz = ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_void_p, ctypes.c_size_t
        L.jetlong_group_size.restype = i64
        L.jetlong_group_size.argtypes = [i64, i64]
        L.jetlong_workspace_bytes.restype = sz
        L.jetlong_workspace_bytes.argtypes = [i32, i64, i32, i32, i32, i32]
        tail = [i64, i32, i32, i32, i64, i64, dbl, i32, vp, sz, vp]
        L.jetlong_prefill.restype = i32
        L.jetlong_prefill.argtypes = [vp] * 5 + tail
        L.jetlong_prefill_prerotated.restype = i32
        L.jetlong_prefill_prerotated.argtypes = [vp] * 5 + tail
        L.jetlong_prefill_unfused.restype = i32
        L.jetlong_prefill_unfused.argtypes = [vp] * 5 + tail
        L.jetlong_prefill_opt.restype = i32
        L.jetlong_prefill_opt.argtypes = [vp] * 5 + tail + [vp]
        L.jetlong_prefill_prerotated_opt.restype = i32
        L.jetlong_prefill_prerotated_opt.argtypes = [vp] * 5 + tail + [vp]
        L.jetlong_host_release.restype = None
        L.jetlong_decode_paged_workspace_bytes.restype = sz
        L.jetlong_decode_paged_workspace_bytes.argtypes = [i64, i32, i32, i32, i32]
        L.jetlong_decode_paged.restype = i32
        L.jetlong_decode_paged.argtypes = [vp, vp, vp, vp, vp, i32, i32, i64, vp, vp, i32, i32, i32, i64, i64, dbl, i32, vp, sz, vp]
        L.jetlong_decode_opt.restype = i32
        L.jetlong_decode_opt.argtypes = [vp] * 5 + tail + [vp]
        L.jetlong_decode.restype = i32
        L.jetlong_decode.argtypes = [vp] * 5 + tail
        L.jetlong_decode_static.restype = i32
        L.jetlong_decode_static.argtypes = [vp] * 5 + [i64, i32, i32, i32, i64, i64, dbl, i32, vp]
        L.jetlong_decode_static_init.restype = i32
        L.jetlong_decode_static_init.argtypes = []
        ctail = [i64, i32, i32, i32, i32, vp, sz, vp]
        L.jetlong_causal_prefill.restype = i32
        L.jetlong_causal_prefill.argtypes = [vp] * 5 + ctail
        L.jetlong_causal_decode.restype = i32
        L.jetlong_causal_decode.argtypes = [vp] * 5 + ctail
        L.jetlong_prefill_host.restype = i32
        L.jetlong_prefill_host.argtypes = [vp] * 5 + [i64, i32, i32, i32, i64, i64, dbl, i32]
        L.jetlong_status_string.restype = ctypes.c_char_p
        L.jetlong_status_string.argtypes = [i32]
        L.jetlong_launch_count.restype = i64
        L.jetlong_set_prefill_impl.restype = i32
        L.jetlong_set_prefill_impl.argtypes = [i32]
        L.jetlong_prefill_uses_umma.restype = i32
        L.jetlong_prefill_uses_umma.argtypes = [i64, i32, i32, i32]
        L.jetlong_set_prefill_precision.restype = i32
        L.jetlong_set_prefill_precision.argtypes = [i32]
        _lib = L
    return _lib


def _check(rc):
    if rc != OK:
        raise JetlongError(rc, lib().jetlong_status_string(rc).decode())


def _dt(t):
    if t.dtype == torch.bfloat16:
        return BF16
    if t.dtype == torch.float32:
        return FP32
    raise TypeError("libjetlong takes bf16 or fp32 tensors, got %s" % t.dtype)


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def jetlong_group_size(L, w_pretrained):
    return int(lib().jetlong_group_size(int(L), int(w_pretrained)))


def jetlong_workspace_bytes(op, L, H_q, H_kv, head_dim, dtype):
    return int(lib().jetlong_workspace_bytes(op, int(L), H_q, H_kv, head_dim, dtype))


def jetlong_launch_count():
    return int(lib().jetlong_launch_count())


def jetlong_set_prefill_impl(impl):
    return int(lib().jetlong_set_prefill_impl(int(impl)))


def jetlong_set_prefill_precision(mode):
    return int(lib().jetlong_set_prefill_precision(int(mode)))


def alloc_workspace(op, L, H_q, H_kv, head_dim, dtype, device="cuda"):
    n = jetlong_workspace_bytes(op, L, H_q, H_kv, head_dim, dtype)
    return torch.zeros(max(n, 256), dtype=torch.uint8, device=device)


def _prefill_args(Q, K, V, out, lse):
    assert Q.is_cuda and K.is_cuda and V.is_cuda and Q.is_contiguous() and K.is_contiguous() and V.is_contiguous()
    L, H_q, d = Q.shape
    assert K.shape == V.shape and K.shape[0] == L and K.shape[2] == d and K.dtype == Q.dtype == V.dtype
    H_kv = K.shape[1]
    if out is None:
        out = torch.empty_like(Q)
    if lse is None:
        lse = torch.empty((H_q, L), dtype=torch.float32, device=Q.device)
    return L, H_q, H_kv, d, out, lse


def jetlong_prefill(Q, K, V, *, w_local, w_pretrained, rope_theta, out=None, lse=None, workspace=None, precision=None,
                    impl=None, remote_map=None, yarn=None):
    """Bifocal prefill.  Q [L,H_q,d], K/V [L,H_kv,d] (bf16 or fp32, RoPE'd at true positions).  Returns out, lse.
    precision / impl: per-call jetlong_options (None = the thread's default)."""
    L, H_q, H_kv, d, out, lse = _prefill_args(Q, K, V, out, lse)
    dt = _dt(Q)
    if workspace is None:
        workspace = alloc_workspace(OP_PREFILL, L, H_q, H_kv, d, dt, Q.device)
    _check(lib().jetlong_prefill_opt(Q.data_ptr(), K.data_ptr(), V.data_ptr(), out.data_ptr(), lse.data_ptr(), L, H_q,
                                     H_kv, d, int(w_local), int(w_pretrained), float(rope_theta), dt,
                                     workspace.data_ptr(), workspace.numel(), _stream(),
                                     _options(precision, impl, remote_map, yarn)))
    return out, lse


def jetlong_prefill_prerotated(Q, K, V, *, w_local, w_pretrained, rope_theta, out=None, lse=None, workspace=None,
                               precision=None, impl=None, remote_map=None, yarn=None):
    """Workspace variant of the bifocal prefill: K is correction-rotated once into a scratch in the workspace."""
    L, H_q, H_kv, d, out, lse = _prefill_args(Q, K, V, out, lse)
    dt = _dt(Q)
    if workspace is None:
        workspace = alloc_workspace(OP_PREFILL_PREROTATED, L, H_q, H_kv, d, dt, Q.device)
    _check(lib().jetlong_prefill_prerotated_opt(Q.data_ptr(), K.data_ptr(), V.data_ptr(), out.data_ptr(), lse.data_ptr(),
                                                L, H_q, H_kv, d, int(w_local), int(w_pretrained), float(rope_theta), dt,
                                                workspace.data_ptr(), workspace.numel(), _stream(),
                                                _options(precision, impl, remote_map, yarn)))
    return out, lse


def jetlong_prefill_unfused(Q, K, V, *, w_local, w_pretrained, rope_theta, out=None, lse=None, workspace=None):
    """The paper's unfused three-call procedure (A + B - C, Eq.(7)) on the GPU: a baseline, not the product path."""
    L, H_q, H_kv, d, out, lse = _prefill_args(Q, K, V, out, lse)
    dt = _dt(Q)
    if workspace is None:
        workspace = alloc_workspace(OP_PREFILL_UNFUSED, L, H_q, H_kv, d, dt, Q.device)
    _check(lib().jetlong_prefill_unfused(Q.data_ptr(), K.data_ptr(), V.data_ptr(), out.data_ptr(), lse.data_ptr(),
                                         L, H_q, H_kv, d, int(w_local), int(w_pretrained), float(rope_theta), dt,
                                         workspace.data_ptr(), workspace.numel(), _stream()))
    return out, lse


def jetlong_causal_prefill(Q, K, V, *, out=None, lse=None, workspace=None):
    """Matched control: plain causal attention on the given Q, K, V."""
    L, H_q, H_kv, d, out, lse = _prefill_args(Q, K, V, out, lse)
    dt = _dt(Q)
    if workspace is None:
        workspace = alloc_workspace(OP_CAUSAL_PREFILL, L, H_q, H_kv, d, dt, Q.device)
    _check(lib().jetlong_causal_prefill(Q.data_ptr(), K.data_ptr(), V.data_ptr(), out.data_ptr(), lse.data_ptr(), L,
                                        H_q, H_kv, d, dt, workspace.data_ptr(), workspace.numel(), _stream()))
    return out, lse


def _decode_args(q, Kc, Vc, L, out, lse):
    assert q.is_cuda and q.is_contiguous() and Kc.is_contiguous() and Vc.is_contiguous()
    H_q, d = q.shape
    assert Kc.shape == Vc.shape and Kc.shape[0] >= L and Kc.shape[2] == d and Kc.dtype == q.dtype
    H_kv = Kc.shape[1]
    if out is None:
        out = torch.empty_like(q)
    if lse is None:
        lse = torch.empty((H_q,), dtype=torch.float32, device=q.device)
    return H_q, H_kv, d, out, lse


def jetlong_decode(q, Kcache, Vcache, L, *, w_local, w_pretrained, rope_theta, out=None, lse=None, workspace=None,
                   remote_map=None, yarn=None):
    """Bifocal decode of the query at position L-1 against cache rows 0..L-1.  q [H_q,d]."""
    H_q, H_kv, d, out, lse = _decode_args(q, Kcache, Vcache, L, out, lse)
    dt = _dt(q)
    if workspace is None:
        workspace = alloc_workspace(OP_DECODE, L, H_q, H_kv, d, dt, q.device)
    _check(lib().jetlong_decode_opt(q.data_ptr(), Kcache.data_ptr(), Vcache.data_ptr(), out.data_ptr(), lse.data_ptr(),
                                    int(L), H_q, H_kv, d, int(w_local), int(w_pretrained), float(rope_theta), dt,
                                    workspace.data_ptr(), workspace.numel(), _stream(),
                                    _options(remote_map=remote_map, yarn=yarn)))
    return out, lse


STATIC_SCRATCH_BYTES = 8 << 20


def jetlong_decode_static_init():
    """Resolve the device address of the library's static scratch for the current device (optional; see jetlong.h)."""
    _check(lib().jetlong_decode_static_init())


def jetlong_decode_static(q, Kcache, Vcache, L, *, w_local, w_pretrained, rope_theta, out, lse):
    """jetlong_decode without any allocation: no workspace argument (the scratch is a static device array inside the
    library, at most STATIC_SCRATCH_BYTES), and `out` / `lse` must be given.  Calls that overlap on the GPU race."""
    H_q, H_kv, d, out, lse = _decode_args(q, Kcache, Vcache, L, out, lse)
    _check(lib().jetlong_decode_static(q.data_ptr(), Kcache.data_ptr(), Vcache.data_ptr(), out.data_ptr(), lse.data_ptr(),
                                       int(L), H_q, H_kv, d, int(w_local), int(w_pretrained), float(rope_theta), _dt(q),
                                       _stream()))
    return out, lse


def jetlong_causal_decode(q, Kcache, Vcache, L, *, out=None, lse=None, workspace=None):
    H_q, H_kv, d, out, lse = _decode_args(q, Kcache, Vcache, L, out, lse)
    dt = _dt(q)
    if workspace is None:
        workspace = alloc_workspace(OP_CAUSAL_DECODE, L, H_q, H_kv, d, dt, q.device)
    _check(lib().jetlong_causal_decode(q.data_ptr(), Kcache.data_ptr(), Vcache.data_ptr(), out.data_ptr(),
                                       lse.data_ptr(), int(L), H_q, H_kv, d, dt, workspace.data_ptr(),
                                       workspace.numel(), _stream()))
    return out, lse


def jetlong_prefill_host(Q, K, V, *, w_local, w_pretrained, rope_theta, out=None, lse=None):
    """End-to-end call with HOST tensors (pinned or pageable): H2D, prefill, D2H inside the library."""
    assert not Q.is_cuda and Q.is_contiguous() and K.is_contiguous() and V.is_contiguous()
    L, H_q, d = Q.shape
    H_kv = K.shape[1]
    if out is None:
        out = torch.empty_like(Q)
    if lse is None:
        lse = torch.empty((H_q, L), dtype=torch.float32)
    _check(lib().jetlong_prefill_host(Q.data_ptr(), K.data_ptr(), V.data_ptr(), out.data_ptr(), lse.data_ptr(), L, H_q,
                                      H_kv, d, int(w_local), int(w_pretrained), float(rope_theta), _dt(Q)))
    return out, lse


def jetlong_decode_paged(q, Kpool, Vpool, page_table, seq_lens, *, w_local, w_pretrained, rope_theta, out=None, lse=None,
                         workspace=None):
    """Batched decode over a paged cache.  q [B,H_q,d]; Kpool/Vpool [pages*128,H_kv,d]; page_table int32 [B,max_pages] on the
    device; seq_lens: a sequence of B ints (host)."""
    assert q.is_cuda and q.is_contiguous() and Kpool.is_contiguous() and Vpool.is_contiguous()
    assert page_table.is_cuda and page_table.dtype == torch.int32 and page_table.is_contiguous()
    Bn, H_q, d = q.shape
    H_kv = Kpool.shape[1]
    assert Kpool.shape == Vpool.shape and Kpool.shape[0] % 128 == 0 and page_table.shape[0] == Bn and len(seq_lens) == Bn
    if out is None:
        out = torch.empty_like(q)
    if lse is None:
        lse = torch.empty((Bn, H_q), dtype=torch.float32, device=q.device)
    lens = (ctypes.c_int64 * Bn)(*[int(x) for x in seq_lens])
    if workspace is None:
        n = int(lib().jetlong_decode_paged_workspace_bytes(max(int(x) for x in seq_lens), Bn, H_q, H_kv, d))
        workspace = torch.zeros(max(n, 256), dtype=torch.uint8, device=q.device)
    _check(lib().jetlong_decode_paged(q.data_ptr(), Kpool.data_ptr(), Vpool.data_ptr(), page_table.data_ptr(), lens, Bn,
                                      page_table.shape[1], Kpool.shape[0] // 128, out.data_ptr(), lse.data_ptr(), H_q, H_kv, d,
                                      int(w_local), int(w_pretrained), float(rope_theta), _dt(q), workspace.data_ptr(),
                                      workspace.numel(), _stream()))
    return out, lse
