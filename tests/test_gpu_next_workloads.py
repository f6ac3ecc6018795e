"""second workloads on the same kernels, sampled rows against the fp64 oracle.

  - Llama-3-shaped: w_pretrained = 8192, rope_theta = 5e5, L = 131072 -> G = 16: a large-G stress of the
    two-level rotation table (Delta reaches -122880) and of the in-row recurrence (n stalls once every 16 keys).
  - 256K-native: w_pretrained = 262144, L = 524288 -> G = 2 (Table 3); head counts are not in the paper, a small
    GQA shape keeps the test short.  L = 524288 is also the longest sequence any test runs (4096 key tiles per row block).
Inputs follow the DESIGN.md recipe (N(0,1), 4 outlier K channels x8, RoPE at true positions in fp64, one bf16 rounding).
"""
import pytest
import torch

import paper_2607_07740_b200 as J
from paper_2607_07740_b200 import workloads as W

from parity_util import check, gather, oracle_rows

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _sampled(fn, L, H_q, H_kv, theta, w_pre, w0, seed, n_pairs, what):
    Q, K, V = W.make_qkv(L, H_q, H_kv, 128, theta, "bf16", seed, True, DEV)
    out, lse = fn(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    torch.cuda.synchronize()
    G = J.jetlong_group_size(L, w_pre)
    rows, heads = W.sample_pairs(L, H_q, n_pairs, seed, w0, G)
    ro, rl = oracle_rows(Q, K, V, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    return check(*gather(out, lse, rows, heads), ro, rl, Q.dtype, what)


@pytest.mark.parametrize("fn", [J.jetlong_prefill, J.jetlong_prefill_prerotated], ids=["on_the_fly", "prerotated"])
def test_llama3_shaped_G16_prefill(fn):
    assert J.jetlong_group_size(131072, 8192) == 16
    _sampled(fn, 131072, 8, 2, 5e5, 8192, 4096, 7740801, 96, "Llama-3-shaped G=16 L=131072")


def test_llama3_shaped_G16_decode():
    L, H_q, H_kv, theta, w_pre, w0 = 131072, 8, 2, 5e5, 8192, 4096
    Q, K, V = W.make_qkv(L, H_q, H_kv, 128, theta, "bf16", 7740802, True, DEV, q_pos0=L - 1, n_q=1)
    out, lse = J.jetlong_decode(Q[0].contiguous(), K, V, L, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    torch.cuda.synchronize()
    import numpy as np
    heads = np.arange(H_q, dtype=np.int32)
    rows = np.full(H_q, L - 1, dtype=np.int64)
    ro, rl = oracle_rows(Q, K, V, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=theta,
                         q_pos_rows=np.zeros(H_q, dtype=np.int64))
    check(out, lse, ro, rl, Q.dtype, "Llama-3-shaped G=16 decode")


@pytest.mark.parametrize("fn", [J.jetlong_prefill, J.jetlong_prefill_prerotated], ids=["on_the_fly", "prerotated"])
def test_256k_native_512k_prefill(fn):
    assert J.jetlong_group_size(524288, 262144) == 2
    _sampled(fn, 524288, 4, 2, 1e6, 262144, 4096, 7740803, 48, "256K-native G=2 L=524288")


def test_256k_native_1m_prefill_and_decode():
    """Table 3: the 256K-native model at L = 1048576 -> G = 4, the longest length the paper reports.  One CTA pair walks
    8192 key tiles; the rotation table reaches n = 786432.  Prefill on sampled rows, then one decode step at the same L."""
    import numpy as np
    L, H_q, H_kv, theta, w_pre, w0 = 1048576, 2, 1, 1e6, 262144, 4096
    assert J.jetlong_group_size(L, w_pre) == 4
    Q, K, V = W.make_qkv(L, H_q, H_kv, 128, theta, "bf16", 7740804, True, DEV)
    out, lse = J.jetlong_prefill(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    torch.cuda.synchronize()
    rows, heads = W.sample_pairs(L, H_q, 24, 7740804, w0, 4)
    ro, rl = oracle_rows(Q, K, V, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    check(*gather(out, lse, rows, heads), ro, rl, Q.dtype, "256K-native G=4 L=1048576")
    od, ld = J.jetlong_decode(Q[L - 1].contiguous(), K, V, L, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    torch.cuda.synchronize()
    hh = np.arange(H_q, dtype=np.int32)
    rr = np.full(H_q, L - 1, dtype=np.int64)
    do, dl = oracle_rows(Q, K, V, rr, hh, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    check(od, ld, do, dl, Q.dtype, "256K-native G=4 decode at L=1048576")
