"""Seeded synthetic inputs for the Jet-Long bifocal-attention hot path.

This module serves BOTH the CUDA path and the CPU oracle (the same tensors are handed to each), so it
holds none of the method's arithmetic: no group size, no remote map, no correction rotation, no
softmax.  It only draws N(0,1) activations, optionally scales a few key channels ("outlier channels",
BASELINE.json configs 2-5), applies standard RoPE at the TRUE absolute positions in fp64 (the input
contract of Eq.(4) P:97 and q_local in Eq.(6)) and rounds once to the input dtype.

The recipe stands in for the paper's Qwen3-1.7B/4B/8B activations on RULER/HELMET/PG-19 prompts
(P:123), which need weights and datasets that are not available offline.
"""
from dataclasses import dataclass

import torch

SEED_BASE = 7740 * 1000


@dataclass(frozen=True)
class Config:
    """One BASELINE.json configuration (shapes only)."""
    name: str
    dtype: str          # "bf16" | "fp32"
    L: int
    H_q: int
    H_kv: int
    d: int
    rope_theta: float
    w_pretrained: int
    w_local: int
    outliers: bool
    index: int          # used in the seed

    def seed(self, layer=0):
        return SEED_BASE + 100 * self.index + layer


# BASELINE.json `configs` (index 1..5 as in SURVEY.md 8(d))
C1 = Config("c1_tiny_fp32", "fp32", 1024, 4, 2, 64, 1e4, 256, 64, False, 1)
C2 = Config("c2_qwen3_1p7b_64k", "bf16", 65536, 16, 8, 128, 1e6, 32768, 4096, True, 2)
C3 = Config("c3_qwen3_4b_128k", "bf16", 131072, 32, 8, 128, 1e6, 32768, 4096, True, 3)
C4 = Config("c4_qwen3_8b_stack_128k", "bf16", 131072, 32, 8, 128, 1e6, 32768, 4096, True, 4)
C5 = Config("c5_qwen3_8b_decode", "bf16", 131072, 32, 8, 128, 1e6, 32768, 4096, True, 5)
C3_SWEEP_L = (32768, 32769, 65536, 98304, 131072)
C4_LAYERS = 36
C4_W_LOCAL = (2048, 4096, 8192)
C5_L0 = (65536, 131072)
C5_STEPS = 256


def torch_dtype(name):
    return {"bf16": torch.bfloat16, "fp32": torch.float32}[name]


def _rope_true_positions(x, pos0, theta, chunk=8192):
    """Standard half-split RoPE of x[n, H, d] (fp64) at positions pos0 .. pos0+n-1, in place."""
    n, H, d = x.shape
    h = d // 2
    inv = theta ** (-2.0 * torch.arange(h, dtype=torch.float64, device=x.device) / d)
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        pos = torch.arange(pos0 + s, pos0 + e, dtype=torch.float64, device=x.device)
        ang = pos[:, None] * inv[None, :]
        c = torch.cos(ang)[:, None, :]
        sn = torch.sin(ang)[:, None, :]
        a = x[s:e, :, :h].clone()
        b = x[s:e, :, h:]
        x[s:e, :, :h] = a * c - b * sn
        x[s:e, :, h:] = a * sn + b * c
    return x


def make_qkv(L, H_q, H_kv, d, rope_theta, dtype, seed, outliers=False, device="cpu", q_pos0=0, n_q=None, k_pos0=0,
             profile=None):
    """Q [n_q,H_q,d], K [L,H_kv,d], V [L,H_kv,d] in `dtype` on `device`.

    Q rows sit at absolute positions q_pos0 .. q_pos0+n_q-1 (default: 0..L-1); K rows at k_pos0 .. k_pos0+L-1
    (default 0..L-1; a non-zero k_pos0 is only used by the global-rotation invariance test).
    outliers: 4 seeded channel indices per KV head of the un-rotated x_k are scaled by 8.
    profile (stress inputs for the precision-margin tests; value distributions only, no method arithmetic):
      "switch"     the outlier channels change halfway through the sequence (4 channels x8 on rows < L/2, 4 others on the rest)
      "q_outliers" the 4 loud channels are in the un-rotated x_q (per query head) instead of x_k
      "loud"       every channel of x_k x1.5 on top of the standard outlier channels
      "slow_pairs" the loud channels are the frequency pairs 32 and 33 (channels d/4, d/4+1 and their partners), x8 in x_k and
                   x4 in x_q: the stress input of the decode kernel's second-order treatment of the slow pairs
    """
    n_q = L if n_q is None else n_q
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(int(seed))
    td = torch_dtype(dtype) if isinstance(dtype, str) else dtype
    xq = torch.randn((n_q, H_q, d), generator=gen, device=dev, dtype=torch.float32).double()
    xk = torch.randn((L, H_kv, d), generator=gen, device=dev, dtype=torch.float32).double()
    v = torch.randn((L, H_kv, d), generator=gen, device=dev, dtype=torch.float32)
    if profile == "switch":
        for kv in range(H_kv):
            idx = torch.randperm(d, generator=gen, device=dev)[:8]
            xk[: L // 2, kv, idx[:4]] *= 8.0
            xk[L // 2:, kv, idx[4:]] *= 8.0
    elif profile == "q_outliers":
        for h in range(H_q):
            idx = torch.randperm(d, generator=gen, device=dev)[:4]
            xq[:, h, idx] *= 8.0
    elif profile == "slow_pairs":
        idx = torch.tensor([d // 4, d // 4 + 1, d // 4 + d // 2, d // 4 + 1 + d // 2], device=dev)
        xk[:, :, idx] *= 8.0
        xq[:, :, idx] *= 4.0
    elif outliers or profile == "loud":
        for kv in range(H_kv):
            idx = torch.randperm(d, generator=gen, device=dev)[:4]
            xk[:, kv, idx] *= 8.0
        if profile == "loud":
            xk *= 1.5
    Q = _rope_true_positions(xq, q_pos0, rope_theta).to(td).contiguous()
    del xq
    K = _rope_true_positions(xk, k_pos0, rope_theta).to(td).contiguous()
    del xk
    return Q, K, v.to(td).contiguous()


def make_config_inputs(cfg, device="cpu", layer=0, L=None):
    L = cfg.L if L is None else L
    return make_qkv(L, cfg.H_q, cfg.H_kv, cfg.d, cfg.rope_theta, cfg.dtype, cfg.seed(layer), cfg.outliers, device)


def make_decode_inputs(cfg, L0, steps, device="cpu"):
    """Decode workload (config 5): a cache of L0+steps-1 rows and one query per step.

    Step t (0-based) runs at L = L0 + t: the cache holds rows 0..L-1 (the current token included,
    P:73) and the query q_t sits at position L-1.  Returns Qsteps [steps,H_q,d], Kcache, Vcache.
    """
    Ltot = L0 + steps - 1
    return make_qkv(Ltot, cfg.H_q, cfg.H_kv, cfg.d, cfg.rope_theta, cfg.dtype, cfg.seed(L0 // 65536), cfg.outliers,
                    device, q_pos0=L0 - 1, n_q=steps)


def sample_pairs(L, H_q, n, seed, w_local=None, G=None):
    """n seeded random (row, head) pairs plus fixed edge rows (SURVEY.md 8(c) 'Large configs')."""
    gen = torch.Generator()
    gen.manual_seed(int(seed) + 17)
    rows = torch.randint(0, L, (n,), generator=gen).tolist()
    heads = torch.randint(0, H_q, (n,), generator=gen).tolist()
    edge = [0, 127, 128, L - 1, L - 2]
    if w_local is not None:
        edge += [w_local - 1, w_local, w_local + 1, w_local + 127, w_local + 128, w_local + 129]
    if G is not None and G > 1:
        edge += [G - 1, G, L - 1 - ((L - 1) % G), L - 1 - ((L - 1) % G) - 1]
    edge += [L // 2 - 1, L // 2, (L // 128) * 128 - 1, (L // 128) * 128]
    for i, r in enumerate(edge):
        if 0 <= r < L:
            rows.append(int(r))
            heads.append(i % H_q)
    return rows, heads
