"""jetlong_decode_static: the allocation-free decode entry point (include/jetlong.h) against the existing jetlong_decode path.

Collected last on purpose (the file name sorts after every other test file): the suite runs with `pytest -x`, a failure here
must not hide other tests.  The test passes alone in a fresh process (the first call resolves the scratch address itself) and
after the other tests (the static scratch then holds whatever earlier calls left: the entry point must not depend on it).
"""
import ctypes

import pytest
import torch

import paper_2607_07740_b200 as J
from paper_2607_07740_b200 import binding as B
from paper_2607_07740_b200 import workloads as W

from parity_util import TOL

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _close(o_new, l_new, o_ref, l_ref, what):
    tol = TOL[torch.bfloat16]
    eo = (o_new.float() - o_ref.float()).abs().max().item()
    el = (l_new - l_ref).abs().max().item()
    rel = ((o_new.float() - o_ref.float()).norm() / o_ref.float().norm()).item()
    assert eo <= tol["out_abs"] and rel <= tol["out_rel"] and el <= tol["lse"], (what, eo, rel, el)
    assert torch.isfinite(o_new.float()).all() and torch.isfinite(l_new).all(), what
    return eo, el


def test_decode_static_matches_decode_on_two_calls_in_a_row():
    """Config-5 head layout (H_q / H_kv = 32 / 8, d = 128, bf16).  Call 1 at L = 20000 (G = 5), call 2 right behind it on the
    same stream at L + 1 with the next query (the scratch keeps call 1's tables and partials), call 3 at another length and
    window (tables rebuilt, partials at another offset).  Each against jetlong_decode with a caller workspace."""
    H_q, H_kv, d, theta, w_pre, w0 = 32, 8, 128, 1e6, 4096, 512
    L = 20000
    Qs, Kc, Vc = W.make_qkv(L + 1, H_q, H_kv, d, theta, "bf16", 8842, True, DEV, q_pos0=L - 1, n_q=2)
    assert J.jetlong_group_size(L, w_pre) == 5
    kw = dict(w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    ref = [J.jetlong_decode(Qs[t].contiguous(), Kc, Vc, L + t, **kw) for t in range(2)]
    torch.cuda.synchronize()
    # outputs are allocated by the caller, before the calls; poisoned so that a call that writes nothing is seen
    outs = [torch.full((H_q, d), float("nan"), dtype=torch.bfloat16, device=DEV) for _ in range(3)]
    lses = [torch.full((H_q,), float("nan"), dtype=torch.float32, device=DEV) for _ in range(3)]
    qs = [Qs[t].contiguous() for t in range(2)]
    torch.cuda.synchronize()
    mem0 = torch.cuda.memory_allocated()
    for t in range(2):                                               # two calls in a row, no synchronisation in between
        J.jetlong_decode_static(qs[t], Kc, Vc, L + t, out=outs[t], lse=lses[t], **kw)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == mem0                     # the binding allocated nothing either
    for t in range(2):
        eo, el = _close(outs[t], lses[t], ref[t][0], ref[t][1], "call %d" % (t + 1))
        # same kernels, same split plan, same table values: the two paths agree to the bit
        assert torch.equal(outs[t], ref[t][0]) and torch.equal(lses[t], ref[t][1]), (t, eo, el)
    # a different shape of the same cache afterwards: shorter length, other window -> other table rows, other partial offset
    L3, w3 = 7777, 100
    q3 = W.make_qkv(L3, H_q, H_kv, d, theta, "bf16", 8843, True, DEV, q_pos0=L3 - 1, n_q=1)[0][0].contiguous()
    r3 = J.jetlong_decode(q3, Kc, Vc, L3, w_local=w3, w_pretrained=2048, rope_theta=theta)
    J.jetlong_decode_static(q3, Kc, Vc, L3, w_local=w3, w_pretrained=2048, rope_theta=theta, out=outs[2], lse=lses[2])
    torch.cuda.synchronize()
    _close(outs[2], lses[2], r3[0], r3[1], "call 3")
    # and the first shape again: the tables of call 3 are in the scratch now
    J.jetlong_decode_static(qs[0], Kc, Vc, L, out=outs[0], lse=lses[0], **kw)
    torch.cuda.synchronize()
    _close(outs[0], lses[0], ref[0][0], ref[0][1], "call 4")


def test_decode_static_rejects_what_the_scratch_cannot_hold():
    lib = B.lib()
    H_q, H_kv, d = 32, 8, 128
    q = torch.zeros((H_q, d), dtype=torch.bfloat16, device=DEV)
    kv = torch.zeros((128, H_kv, d), dtype=torch.bfloat16, device=DEV)
    out = torch.zeros_like(q)
    lse = torch.zeros((H_q,), dtype=torch.float32, device=DEV)
    L_big = 1 << 24                                                    # tables alone: 65537 rows x 512 B = 33.6 MB
    assert J.jetlong_workspace_bytes(B.OP_DECODE, L_big, H_q, H_kv, d, B.BF16) > B.STATIC_SCRATCH_BYTES
    n0 = J.jetlong_launch_count()
    rc = lib.jetlong_decode_static(q.data_ptr(), kv.data_ptr(), kv.data_ptr(), out.data_ptr(), lse.data_ptr(), L_big, H_q, H_kv,
                                   d, 4096, 32768, 1e6, B.BF16, None)
    assert rc == 4 and J.jetlong_launch_count() == n0                  # JETLONG_SCRATCH_EXCEEDED, nothing launched
    assert b"JETLONG_STATIC_SCRATCH_BYTES" in lib.jetlong_status_string(rc)
    # the same limit the header states: the largest L of the config-5 layout that fits is above 1.5 M rows
    assert J.jetlong_workspace_bytes(B.OP_DECODE, 1500000, H_q, H_kv, d, B.BF16) <= B.STATIC_SCRATCH_BYTES
    # invalid arguments are still reported as such
    rc = lib.jetlong_decode_static(None, kv.data_ptr(), kv.data_ptr(), out.data_ptr(), lse.data_ptr(), 100, H_q, H_kv, d, 16, 64,
                                   1e6, B.BF16, None)
    assert rc == 1
    J.jetlong_decode_static_init()                                     # idempotent
