"""the frequency-interpolation remote map (Section 4.7; R17) on the GPU against its
oracle routine (oracle.attend_rows_freq): every row on small shapes through all three prefill implementations and decode."""
import numpy as np
import pytest
import torch

import oracle
import paper_2607_07740_b200 as J
from paper_2607_07740_b200 import binding as B
from paper_2607_07740_b200 import workloads as W

from parity_util import all_pairs, check, gather

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _oracle(Q, K, V, rows, heads, q_rows=None, **kw):
    Kf, Vf = K.float().cpu().numpy(), V.float().cpu().numpy()
    ri = torch.as_tensor(rows if q_rows is None else q_rows, dtype=torch.long, device=Q.device)
    hi = torch.as_tensor(heads, dtype=torch.long, device=Q.device)
    Qr = Q[ri, hi].float().cpu().numpy()
    return oracle.attend_rows_freq((Qr, Q.shape[1]), Kf, Vf, rows, heads, q_is_compact=True, **kw)


@pytest.mark.parametrize("L,H_q,H_kv,d,theta,w_pre,w0,dtype,impl,yarn", [
    (777, 4, 2, 128, 1e6, 200, 100, "bf16", 4, None),         # two-tile tcgen05 kernel, default ramp (alpha 1, beta 32)
    (1300, 4, 2, 128, 1e4, 300, 64, "bf16", 4, (0.5, 8.0)),   # a ramp that splits the 64 frequencies three ways at this size
    (2200, 8, 2, 128, 1e6, 512, 128, "bf16", 4, None),        # G = 5, g = 4
    (1300, 4, 2, 128, 1e4, 300, 64, "bf16", 1, (0.5, 8.0)),   # one-tile kernel
    (600, 4, 2, 64, 1e4, 128, 16, "fp32", 0, (0.5, 8.0)),     # SIMT fp32: the tight tolerance pins the map itself
    (300, 3, 1, 128, 1e6, 100, 7, "fp32", 0, None),
])
def test_freq_map_prefill_full_rows(L, H_q, H_kv, d, theta, w_pre, w0, dtype, impl, yarn):
    Q, K, V = W.make_qkv(L, H_q, H_kv, d, theta, dtype, 8800 + L, dtype == "bf16", DEV)
    out, lse = J.jetlong_prefill(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=theta, impl=impl,
                                 remote_map=B.MAP_FREQ_INTERP, yarn=yarn)
    torch.cuda.synchronize()
    rows, heads = all_pairs(L, H_q)
    a, b = yarn if yarn else (1.0, 32.0)
    ro, rl = _oracle(Q, K, V, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=theta, alpha=a, beta=b)
    check(*gather(out, lse, rows, heads), ro, rl, Q.dtype, "freq map L=%d impl %d" % (L, impl))
    # and it is a different function from aliasing (so the test cannot pass by ignoring the option)
    oa, la = J.jetlong_prefill(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=theta, impl=impl)
    assert (la - lse).abs().max() > 1e-2


def test_freq_map_prerotated_and_decode():
    L, H_q, H_kv, theta, w_pre, w0 = 3000, 8, 2, 1e6, 700, 256
    Q, K, V = W.make_qkv(L, H_q, H_kv, 128, theta, "bf16", 8901, True, DEV)
    out, lse = J.jetlong_prefill_prerotated(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=theta, remote_map=B.MAP_FREQ_INTERP)
    rows, heads = all_pairs(L, H_q)
    sel = np.random.RandomState(3).choice(len(rows), 2000, replace=False)
    rows, heads = rows[sel], heads[sel]
    ro, rl = _oracle(Q, K, V, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    check(*gather(out, lse, rows, heads), ro, rl, Q.dtype, "freq map, workspace variant")
    od, ld = J.jetlong_decode(Q[L - 1].contiguous(), K, V, L, w_local=w0, w_pretrained=w_pre, rope_theta=theta,
                              remote_map=B.MAP_FREQ_INTERP)
    torch.cuda.synchronize()
    hh = np.arange(H_q, dtype=np.int32)
    do, dl = _oracle(Q, K, V, np.full(H_q, L - 1, dtype=np.int64), hh, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    check(od, ld, do, dl, Q.dtype, "freq map decode")
    # a following aliasing call on the same workspace must rebuild the tables (the header records the map)
    ws = B.alloc_workspace(B.OP_DECODE, L, H_q, H_kv, 128, B.BF16, DEV)
    J.jetlong_decode(Q[L - 1].contiguous(), K, V, L, w_local=w0, w_pretrained=w_pre, rope_theta=theta, workspace=ws,
                     remote_map=B.MAP_FREQ_INTERP)
    o2, l2 = J.jetlong_decode(Q[L - 1].contiguous(), K, V, L, w_local=w0, w_pretrained=w_pre, rope_theta=theta, workspace=ws)
    o3, l3 = J.jetlong_decode(Q[L - 1].contiguous(), K, V, L, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    assert torch.equal(o2, o3) and torch.equal(l2, l3)


def test_freq_map_G1_is_the_control_bitwise():
    L = 500
    Q, K, V = W.make_qkv(L, 4, 2, 128, 1e6, "bf16", 8902, True, DEV)
    out, lse = J.jetlong_prefill(Q, K, V, w_local=64, w_pretrained=1024, rope_theta=1e6, remote_map=B.MAP_FREQ_INTERP)
    oc, lc = J.jetlong_causal_prefill(Q, K, V)
    assert torch.equal(out, oc) and torch.equal(lse, lc)
