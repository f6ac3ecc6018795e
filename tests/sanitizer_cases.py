"""Small hot-path cases for compute-sanitizer: config 1, two bf16 prefills on the tcgen05 two-tile
kernel (ragged L = 777; a longer one with local, straddle and remote phases), the control, and one decode step.

    compute-sanitizer --tool memcheck|synccheck|racecheck python tests/sanitizer_cases.py [L_long]

Not a pytest module (no test_ prefix): it only runs the calls and checks the results are finite; parity is tests/test_gpu_*.
"""
import os
import sys

import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import paper_2607_07740_b200 as J  # noqa: E402
from paper_2607_07740_b200 import workloads as W  # noqa: E402

L_long = int(sys.argv[1]) if len(sys.argv) > 1 else 8320
dev = "cuda:0"
c = W.C1
Q, K, V = W.make_qkv(c.L, c.H_q, c.H_kv, c.d, c.rope_theta, "fp32", c.seed(), False, dev)
o, l = J.jetlong_prefill(Q, K, V, w_local=c.w_local, w_pretrained=c.w_pretrained, rope_theta=c.rope_theta)
assert torch.isfinite(o).all() and torch.isfinite(l).all()
print("config 1 ok")
for L, w_pre, w0 in ((777, 200, 100), (L_long, max(L_long // 4, 64), 256)):
    Q, K, V = W.make_qkv(L, 4, 2, 128, 1e6, "bf16", 1234 + L, True, dev)
    o, l = J.jetlong_prefill(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=1e6)
    oc, lc = J.jetlong_causal_prefill(Q, K, V)
    torch.cuda.synchronize()
    assert torch.isfinite(o.float()).all() and torch.isfinite(l).all() and torch.isfinite(oc.float()).all()
    print("bf16 prefill L=%d ok" % L)
L = 3000
Q, K, V = W.make_qkv(L, 32, 8, 128, 1e6, "bf16", 77, True, dev, q_pos0=L - 1, n_q=1)
o, l = J.jetlong_decode(Q[0].contiguous(), K, V, L, w_local=512, w_pretrained=1024, rope_theta=1e6)
torch.cuda.synchronize()
assert torch.isfinite(o.float()).all() and torch.isfinite(l).all()
print("decode ok")
