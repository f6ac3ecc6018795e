"""CPU-only checks of the C-ABI boundary: the library loads, exports every symbol include/jetlong.h declares,
computes Eq.(2) on the host and validates arguments before touching the device."""
import ctypes
import os
import re

import pytest

from paper_2607_07740_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "jetlong.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(jetlong_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported_and_bound():
    names = _declared()
    assert len(names) >= 10
    L = B.lib()
    for n in names:
        assert hasattr(L, n), n
    assert sorted(B.EXPORTS) == names


def test_group_size_host():
    assert B.jetlong_group_size(98304, 32768) == 3 and B.jetlong_group_size(98305, 32768) == 4
    assert B.jetlong_group_size(1, 32768) == 1 and B.jetlong_group_size(32768, 32768) == 1
    assert B.jetlong_group_size(0, 5) == -1 and B.jetlong_group_size(5, 0) == -1
    for m in range(1, 50):
        assert B.jetlong_group_size(m * 4096, 4096) == m and B.jetlong_group_size(m * 4096 + 1, 4096) == m + 1


def test_workspace_sizes():
    assert B.jetlong_workspace_bytes(B.OP_PREFILL, 1024, 4, 2, 64, B.FP32) >= 1024 * 32 * 8
    assert B.jetlong_workspace_bytes(B.OP_DECODE, 131072, 32, 8, 128, B.BF16) > 0
    assert B.jetlong_workspace_bytes(B.OP_DECODE, 131072, 32, 8, 96, B.BF16) == 0       # bad head_dim
    assert B.jetlong_workspace_bytes(99, 1024, 4, 2, 64, B.FP32) == 0


def test_validation_happens_before_any_launch():
    L = B.lib()
    buf = (ctypes.c_char * 4096)()
    a = ctypes.addressof(buf)
    a = (a + 15) & ~15
    ok_args = dict(L=8, H_q=2, H_kv=1, d=64, w0=1, w_pre=4, theta=1e4, dt=B.FP32)

    def call(**kw):
        p = dict(ok_args, **kw)
        ptrs = kw.get("ptrs", [a, a, a, a, a])
        return L.jetlong_prefill(*ptrs, p["L"], p["H_q"], p["H_kv"], p["d"], p["w0"], p["w_pre"], p["theta"], p["dt"],
                                 a, 4096, None)

    assert call(ptrs=[0, a, a, a, a]) == B.INVALID_ARG
    assert call(L=0) == B.INVALID_ARG
    assert call(H_q=3, H_kv=2) == B.INVALID_ARG
    assert call(d=96) == B.INVALID_ARG
    assert call(w0=-1) == B.INVALID_ARG
    assert call(w_pre=0) == B.INVALID_ARG
    assert call(theta=0.0) == B.INVALID_ARG
    assert call(dt=7) == B.INVALID_ARG
    assert call(ptrs=[a + 4, a, a, a, a]) == B.INVALID_ARG
    # workspace too small for the rotation table
    assert L.jetlong_prefill(a, a, a, a, a, 4096, 2, 1, 64, 1, 4, 1e4, B.FP32, a, 16, None) == B.INVALID_ARG
    # valid arguments but no B200 here: the library refuses instead of falling back to the CPU
    import torch
    if not torch.cuda.is_available():
        assert call() == B.UNSUPPORTED
    assert b"invalid" in L.jetlong_status_string(B.INVALID_ARG)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_07740_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "jetlong_oracle" not in txt, f


def test_prefill_precision_switch_is_host_state():
    assert B.jetlong_set_prefill_precision(B.PRECISION_FAST) == B.PRECISION_COMPENSATED       # returns the previous mode
    assert B.jetlong_set_prefill_precision(B.PRECISION_COMPENSATED_F16) == B.PRECISION_FAST
    assert B.jetlong_set_prefill_precision(77) == B.PRECISION_COMPENSATED_F16                  # unknown: unchanged
    assert B.jetlong_set_prefill_precision(B.PRECISION_COMPENSATED) == B.PRECISION_COMPENSATED_F16
    assert B.jetlong_set_prefill_precision(B.PRECISION_COMPENSATED) == B.PRECISION_COMPENSATED


def test_workspace_sizes_of_the_prefill_variants():
    """the workspace variant holds tables + K'hi (2 B) + two e5m2 buffers (1 B each) per key channel
    + the selection scratch; the unfused baseline holds the same region + O_A, O_B, O_C in fp32 (4 B per query channel) + two lse."""
    L, H_q, H_kv, d = 65536, 16, 8, 128
    pre = B.jetlong_workspace_bytes(B.OP_PREFILL_PREROTATED, L, H_q, H_kv, d, B.BF16)
    unf = B.jetlong_workspace_bytes(B.OP_PREFILL_UNFUSED, L, H_q, H_kv, d, B.BF16)
    nk, nq = L * H_kv * d, L * H_q * d
    slack = 1 << 20                                       # two-level rotation table (0.2 MB here) + alignment + selection scratch
    assert 4 * nk <= pre <= 4 * nk + slack
    assert pre + 12 * nq + 8 * L * H_q <= unf <= pre + 12 * nq + 8 * L * H_q + slack
    # shapes the tcgen05 kernel does not serve have no such variants
    assert B.jetlong_workspace_bytes(B.OP_PREFILL_PREROTATED, 1024, 4, 2, 64, B.FP32) == 0
    assert B.jetlong_workspace_bytes(B.OP_PREFILL_UNFUSED, 1024, 3, 1, 64, B.BF16) == 0         # head_dim 64
    assert B.jetlong_workspace_bytes(B.OP_PREFILL_UNFUSED, 1024, 3, 1, 128, B.BF16) > 0         # odd H_q / H_kv is served (round 2)


def test_prefill_variants_validate_before_any_launch():
    L = B.lib()
    buf = (ctypes.c_char * 4096)()
    a = (ctypes.addressof(buf) + 15) & ~15
    for fn in (L.jetlong_prefill_prerotated, L.jetlong_prefill_unfused):
        assert fn(0, a, a, a, a, 256, 2, 1, 128, 1, 64, 1e4, B.BF16, a, 4096, None) == B.INVALID_ARG      # null Q
        assert fn(a, a, a, a, a, 256, 2, 1, 128, -1, 64, 1e4, B.BF16, a, 4096, None) == B.INVALID_ARG     # w_local < 0
        assert fn(a, a, a, a, a, 256, 2, 1, 64, 1, 64, 1e4, B.FP32, a, 4096, None) == B.UNSUPPORTED       # fp32 / d = 64
        assert fn(a, a, a, a, a, 256, 2, 1, 128, 1, 64, 1e4, B.BF16, a, 16, None) == B.INVALID_ARG        # workspace too small


def test_prefill_impl_switch_is_host_state():
    prev = B.jetlong_set_prefill_impl(1)                  # the one-tile CTA-pair kernel
    assert B.jetlong_set_prefill_impl(0) == 1
    assert B.jetlong_set_prefill_impl(-1) == 0
    assert B.jetlong_set_prefill_impl(2) == -1            # 2, 3: the removed cluster launches, accepted and mean 1
    assert B.jetlong_set_prefill_impl(prev) == 1


def test_setters_are_per_thread_defaults():
    """The deprecated setters change the CALLING thread's default only (include/jetlong.h: nothing process-global)."""
    import threading
    seen = {}
    prev = B.jetlong_set_prefill_precision(B.PRECISION_FAST)

    def other():
        seen["before"] = B.jetlong_set_prefill_precision(B.PRECISION_COMPENSATED_E5M2)   # a fresh thread starts at the default
        seen["after"] = B.jetlong_set_prefill_precision(B.PRECISION_COMPENSATED)
    th = threading.Thread(target=other)
    th.start()
    th.join()
    assert seen == {"before": B.PRECISION_COMPENSATED, "after": B.PRECISION_COMPENSATED_E5M2}
    assert B.jetlong_set_prefill_precision(prev) == B.PRECISION_FAST                      # untouched by the other thread


def test_options_are_validated_before_any_launch():
    import ctypes
    L = B.lib()
    n0 = B.jetlong_launch_count()
    bad = B.Options(4, B.DEFAULT, B.DEFAULT, B.DEFAULT, 0.0, 0.0)   # struct_bytes too small
    args = [1 << 12] * 5 + [64, 2, 2, 128, 8, 32, 1e4, B.BF16, 1 << 12, 1 << 20, None]
    assert L.jetlong_prefill_opt(*args, ctypes.byref(bad)) == B.INVALID_ARG
    unk = B.Options(ctypes.sizeof(B.Options), 17, B.DEFAULT, B.DEFAULT, 0.0, 0.0)   # unknown precision
    assert L.jetlong_prefill_opt(*args, ctypes.byref(unk)) == B.INVALID_ARG
    bad_map = B.Options(ctypes.sizeof(B.Options), B.DEFAULT, B.DEFAULT, 9, 0.0, 0.0)
    assert L.jetlong_prefill_opt(*args, ctypes.byref(bad_map)) == B.INVALID_ARG
    bad_ramp = B.Options(ctypes.sizeof(B.Options), B.DEFAULT, B.DEFAULT, B.MAP_FREQ_INTERP, 4.0, 2.0)   # beta <= alpha
    assert L.jetlong_prefill_opt(*args, ctypes.byref(bad_ramp)) == B.INVALID_ARG
    assert B.jetlong_launch_count() == n0
