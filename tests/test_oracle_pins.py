"""Pins for the fp64 CPU oracle (oracle/jetlong_oracle.c) against what the paper and the mathematics fix.

None of these compares the oracle with itself through the same code path: each pin is a printed value,
a closed form, an invariant, a library routine (torch SDPA / logsumexp) or an independent formulation
(complex-number RoPE applied from scratch at the remapped positions, Eq.(1)).
"""
import cmath
import math
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2607_07740_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _raw_inputs(L, H_q, H_kv, d, seed):
    g = np.random.default_rng(seed)
    return (g.standard_normal((L, H_q, d)), g.standard_normal((L, H_kv, d)), g.standard_normal((L, H_kv, d)))


def _rope_np(x, pos, theta):
    """Independent numpy RoPE via complex multiplication: z_i = x_i + j x_{i+d/2}, z_i *= exp(j pos theta_i)."""
    L, H, d = x.shape
    h = d // 2
    th = theta ** (-2.0 * np.arange(h) / d)
    z = x[..., :h] + 1j * x[..., h:]
    z = z * np.exp(1j * np.asarray(pos, dtype=np.float64)[:, None, None] * th[None, None, :])
    return np.concatenate([z.real, z.imag], axis=-1)


# ---------------------------------------------------------------- Eq.(2), Eq.(3)
def test_eq2_printed_values():
    n = 0
    for line in open(os.path.join(GOLDEN, "eq2_group_size.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w, L, G, _src = line.split()
        assert oracle.group_size(int(L), int(w)) == int(G), line
        n += 1
    assert n >= 8


@pytest.mark.parametrize("w", [1, 2, 7, 256, 32768, 262144])
def test_eq2_steps_exactly_at_multiples(w):
    for m in range(1, 40):
        assert oracle.group_size(m * w, w) == m
        assert oracle.group_size(m * w + 1, w) == m + 1
        if w > 1:
            assert oracle.group_size(m * w - 1, w) == m
    for L in range(1, w + 1, max(1, w // 13)):
        assert oracle.group_size(L, w) == 1


def test_eq2_eq3_keep_remote_positions_inside_window_and_minimal():
    # "G is the smallest integer that keeps the compressed sequence within the pretrained window"
    rng = np.random.default_rng(0)
    for w in (5, 64, 32768):
        for L in list(rng.integers(1, 40 * w, size=200)) + [w, w + 1, 4 * w, 4 * w + 1]:
            L = int(L)
            G = oracle.group_size(L, w)
            assert oracle.remote_pos(L - 1, G) <= w - 1
            assert oracle.remote_pos(0, G) == 0
            if G > 1:
                assert (L - 1) // (G - 1) > w - 1          # G-1 would overflow the window
            for x in (0, 1, G - 1, G, L - 1):
                assert oracle.remote_pos(x, G) == math.floor(x / G)
                assert oracle.delta(x, G) == math.floor(x / G) - x     # Eq.(5)


# ---------------------------------------------------------------- RoPE / Eq.(6)
def test_rope_d2_by_hand_and_group_law():
    # d = 2, theta_0 = 1: rotating (1, 0) by n gives (cos n, sin n)
    for n in (0, 1, -3, 17):
        y = oracle.rope(np.array([1.0, 0.0]), 1e4, n)
        assert np.allclose(y, [math.cos(n), math.sin(n)], atol=1e-15)
    x = np.random.default_rng(1).standard_normal(64)
    assert np.array_equal(oracle.rope(x, 1e4, 0), x)                       # R_0 = I
    a, b = 1234, -777
    assert np.allclose(oracle.rope(oracle.rope(x, 1e4, a), 1e4, b), oracle.rope(x, 1e4, a + b), atol=1e-12)
    assert abs(np.linalg.norm(oracle.rope(x, 1e6, 98765)) - np.linalg.norm(x)) < 1e-12


@pytest.mark.parametrize("theta,d", [(1e4, 64), (1e6, 128), (5e5, 16)])
def test_rope_matches_input_generator_and_complex_form(theta, d):
    # the oracle's rotation, the generator's RoPE and the complex form agree -> same pairing and sign
    x = np.random.default_rng(2).standard_normal((5, 1, d))
    pos = [0, 1, 77, 4095, 131071]
    ref = _rope_np(x, pos, theta)
    for j, p in enumerate(pos):
        assert np.allclose(oracle.rope(x[j, 0], theta, p), ref[j, 0], atol=1e-10)
    gen = torch.from_numpy(x[:3].copy())
    for j in range(3):
        one = W._rope_true_positions(torch.from_numpy(x[j:j + 1].copy()), pos[j], theta)
        assert np.allclose(one.numpy()[0, 0], ref[j, 0], atol=1e-10)
    del gen


def test_eq6_correction_recovers_remote_phase():
    # R(Delta(k)) RoPE(x, k) = RoPE(x, f(k))  (Eq.(4)-(6) P:97-106), from un-rounded x
    d, theta = 128, 1e6
    x = np.random.default_rng(3).standard_normal(d)
    for G in (2, 3, 4, 5):
        for k in (0, 1, G - 1, G, 4097, 98304, 131071):
            cached = oracle.rope(x, theta, k)
            corrected = oracle.rope(cached, theta, oracle.delta(k, G))
            assert np.allclose(corrected, oracle.rope(x, theta, k // G), atol=1e-10)


# ---------------------------------------------------------------- Eq.(1): closed form
@pytest.mark.parametrize("L,w_pre,w0,d,theta", [(96, 32, 8, 16, 1e4), (70, 16, 0, 8, 100.0), (64, 16, 5, 2, 1e4)])
def test_eq1_closed_form_cosine_sums(L, w_pre, w0, d, theta):
    # every pair (x_i, x_{i+d/2}) = (1, 0): base score = scale * sum_i cos((q-k) th_i),
    # remote score = scale * sum_i cos((f(q)-f(k)) th_i)
    h = d // 2
    x = np.zeros((L, 1, d))
    x[..., :h] = 1.0
    QK = _rope_np(x, np.arange(L), theta)
    G = oracle.group_size(L, w_pre)
    th = theta ** (-2.0 * np.arange(h) / d)
    scale = 1 / math.sqrt(d)
    for q in (0, 1, w0, w0 + 1, L // 2, L - 1):
        s = oracle.scores_row(QK[q, 0], QK, q, 0, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
        for k in range(q + 1):
            rel = (q - k) if q - k <= w0 else (q // G - k // G)
            want = scale * np.cos(rel * th).sum()
            assert abs(s[k] - want) < 5e-6, (q, k)            # inputs were rounded to fp32
        # window edge (R1): k = q - w0 is local, k = q - w0 - 1 is remote ("<=")
    # w0 = 0 leaves only self-attention locally
    s = oracle.scores_row(QK[L - 1, 0], QK, L - 1, 0, w_local=0, w_pretrained=w_pre, rope_theta=theta)
    assert abs(s[L - 1] - scale * h) < 1e-6
    want = scale * np.cos(((L - 1) // G - (L - 2) // G) * th).sum()
    assert abs(s[L - 2] - want) < 5e-6


def test_eq1_from_scratch_complex_bruteforce():
    # Eq.(1) literally: RoPE applied FROM SCRATCH to the content vectors at f(q), f(k) (no correction
    # rotation, no cache), softmax and PV in pure Python -- independent of the oracle's Eq.(6) route.
    L, H_q, H_kv, d, theta, w_pre, w0 = 40, 4, 2, 8, 50.0, 9, 3
    xq, xk, v = _raw_inputs(L, H_q, H_kv, d, 11)
    Q = _rope_np(xq, np.arange(L), theta)
    K = _rope_np(xk, np.arange(L), theta)
    out, lse = oracle.attend_all(Q, K, v, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    G = -(-L // w_pre)
    assert G == 5
    h = d // 2
    th = [theta ** (-2.0 * i / d) for i in range(h)]
    Q32, K32, V32 = Q.astype(np.float32), K.astype(np.float32), v.astype(np.float32)
    for q in range(L):
        for hq in range(H_q):
            kv = hq // (H_q // H_kv)
            s = []
            for k in range(q + 1):
                acc = 0.0
                for i in range(h):
                    # content vectors recovered from the (fp32-rounded) rotated inputs
                    zq = complex(Q32[q, hq, i], Q32[q, hq, i + h]) * cmath.exp(-1j * q * th[i])
                    zk = complex(K32[k, kv, i], K32[k, kv, i + h]) * cmath.exp(-1j * k * th[i])
                    pq, pk = (q, k) if q - k <= w0 else (q // G, k // G)
                    acc += (zq * cmath.exp(1j * pq * th[i]) * (zk * cmath.exp(1j * pk * th[i])).conjugate()).real
                s.append(acc / math.sqrt(d))
            m = max(s)
            p = [math.exp(t - m) for t in s]
            l = sum(p)
            o = [sum(p[k] * float(V32[k, kv, c]) for k in range(q + 1)) / l for c in range(d)]
            assert np.allclose(out[q, hq], o, atol=1e-12)
            assert abs(lse[hq, q] - (m + math.log(l))) < 1e-12


# ---------------------------------------------------------------- G = 1 and the control
@pytest.mark.parametrize("d,theta", [(64, 1e4), (16, 1e6)])
def test_g1_is_bitexact_causal_and_matches_torch_sdpa(d, theta):
    # P:73 "When L <= w_pretrained, f(x) = x and Eq.(1) reduces to the unmodified base attention"
    L, H_q, H_kv = 48, 4, 2
    xq, xk, v = _raw_inputs(L, H_q, H_kv, d, 5)
    Q = _rope_np(xq, np.arange(L), theta).astype(np.float32)
    K = _rope_np(xk, np.arange(L), theta).astype(np.float32)
    V = v.astype(np.float32)
    o_b, l_b = oracle.attend_all(Q, K, V, w_local=7, w_pretrained=L, rope_theta=theta)
    o_c, l_c = oracle.attend_all(Q, K, V, w_local=7, w_pretrained=L, rope_theta=theta, mode="causal")
    assert np.array_equal(o_b, o_c) and np.array_equal(l_b, l_c)
    # library routine: torch SDPA in fp64 with GQA expansion, causal mask, scale 1/sqrt(d)
    tq = torch.from_numpy(Q).double().permute(1, 0, 2)[None]
    tk = torch.from_numpy(K).double().permute(1, 0, 2).repeat_interleave(H_q // H_kv, 0)[None]
    tv = torch.from_numpy(V).double().permute(1, 0, 2).repeat_interleave(H_q // H_kv, 0)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, is_causal=True)[0].permute(1, 0, 2).numpy()
    assert np.allclose(o_c, ref, atol=1e-12)
    sc = (tq[0] @ tk[0].transpose(1, 2)) / math.sqrt(d)
    sc = sc.masked_fill(torch.triu(torch.ones(L, L, dtype=torch.bool), 1), -math.inf)
    assert np.allclose(l_c, torch.logsumexp(sc, -1).numpy(), atol=1e-12)


def test_window_covering_everything_equals_control():
    L, H_q, H_kv, d, theta = 64, 2, 1, 16, 1e4
    xq, xk, v = _raw_inputs(L, H_q, H_kv, d, 6)
    Q = _rope_np(xq, np.arange(L), theta)
    K = _rope_np(xk, np.arange(L), theta)
    for w0 in (L - 1, L, 10 * L):
        o_b, l_b = oracle.attend_all(Q, K, v, w_local=w0, w_pretrained=16, rope_theta=theta)
        o_c, l_c = oracle.attend_all(Q, K, v, w_local=w0, w_pretrained=16, rope_theta=theta, mode="causal")
        assert np.array_equal(o_b, o_c) and np.array_equal(l_b, l_c)
    o_b, _ = oracle.attend_all(Q, K, v, w_local=L - 2, w_pretrained=16, rope_theta=theta)
    assert not np.allclose(o_b[L - 1], o_c[L - 1], atol=1e-6)      # one remote key is enough to differ
    assert np.array_equal(o_b[:L - 1], o_c[:L - 1])


# ---------------------------------------------------------------- Eq.(7)
@pytest.mark.parametrize("L,w_pre,w0,d", [(96, 32, 8, 16), (50, 10, 0, 8), (33, 8, 7, 64), (20, 20, 4, 4), (64, 13, 63, 16)])
def test_eq7_three_call_merge_equals_direct_masking(L, w_pre, w0, d):
    H_q, H_kv, theta = 4, 2, 1e4
    xq, xk, v = _raw_inputs(L, H_q, H_kv, d, 7)
    Q = _rope_np(xq, np.arange(L), theta)
    K = _rope_np(xk, np.arange(L), theta)
    rows = np.repeat(np.arange(L), H_q)
    heads = np.tile(np.arange(H_q), L)
    o_d, l_d = oracle.attend_rows(Q, K, v, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    o_m, l_m, parts = oracle.three_call_rows(Q, K, v, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    assert np.abs(o_d - o_m).max() < 1e-12
    assert np.abs(l_d - l_m).max() < 1e-12
    # rows with no remote key: l_B == l_C exactly, so the subtraction is exactly 0 (R13)
    noremote = rows <= w0
    assert np.array_equal(parts[noremote, 1], parts[noremote, 2])
    assert np.abs(l_m[noremote] - parts[noremote, 0]).max() < 1e-14


# ---------------------------------------------------------------- softmax / PV plumbing
def test_softmax_plumbing_closed_forms():
    L, H_q, H_kv, d, theta = 37, 4, 2, 8, 1e4
    _, xk, v = _raw_inputs(L, H_q, H_kv, d, 8)
    K = _rope_np(xk, np.arange(L), theta).astype(np.float32)
    V = v.astype(np.float32)
    Q0 = np.zeros((L, H_q, d), dtype=np.float32)
    out, lse = oracle.attend_all(Q0, K, V, w_local=3, w_pretrained=8, rope_theta=theta)
    for q in range(L):
        for hq in range(H_q):
            assert np.allclose(out[q, hq], V[:q + 1, hq // 2].astype(np.float64).mean(0), atol=1e-13)
            assert abs(lse[hq, q] - math.log(q + 1)) < 1e-13
    Q = np.random.default_rng(9).standard_normal((L, H_q, d)).astype(np.float32)
    Vc = np.broadcast_to(np.arange(d, dtype=np.float32), (L, H_kv, d)).copy()
    out, _ = oracle.attend_all(Q, K, Vc, w_local=3, w_pretrained=8, rope_theta=theta)
    assert np.allclose(out, Vc[0, 0], atol=1e-12)
    Vh = np.zeros((L, H_kv, d), dtype=np.float32)
    Vh[5, :, 0] = 1.0                                              # one-hot: out[...,0] = p(k=5)
    out, lse = oracle.attend_all(Q, K, Vh, w_local=3, w_pretrained=8, rope_theta=theta)
    s = oracle.scores_row(Q[20, 1], K, 20, 0, w_local=3, w_pretrained=8, rope_theta=theta)
    assert abs(out[20, 1, 0] - math.exp(s[5] - lse[1, 20])) < 1e-13
    assert np.all(out[:5, :, 0] == 0)


# ---------------------------------------------------------------- invariances
def test_shift_invariance():
    L, H_q, H_kv, d, theta, w_pre, w0 = 60, 2, 1, 16, 1e4, 20, 6
    xq, xk, v = _raw_inputs(L, H_q, H_kv, d, 10)
    G = oracle.group_size(L, w_pre)
    assert G == 3
    rows = np.repeat(np.arange(L), H_q)
    heads = np.tile(np.arange(H_q), L)

    def run(c_inputs, c_pos):
        Q = _rope_np(xq, np.arange(L) + c_inputs, theta)
        K = _rope_np(xk, np.arange(L) + c_inputs, theta)
        return oracle.attend_rows(Q, K, v, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=theta, pos_shift=c_pos)

    o0, l0 = run(0, 0)
    # (i) all positions shifted by c: unchanged iff G | c
    o1, l1 = run(15, 15)
    assert np.abs(o0 - o1).max() < 1e-5 and np.abs(l0 - l1).max() < 1e-5       # fp32-rounded inputs
    o2, _ = run(16, 16)
    assert np.abs(o0 - o2).max() > 1e-3
    # (ii) a global rotation R(c) of both Q and K (positions in Eq.(3) unchanged) never matters
    for c in (7, 1000):
        o3, l3 = run(c, 0)
        assert np.abs(o0 - o3).max() < 1e-5 and np.abs(l0 - l3).max() < 1e-5


def test_within_group_aliasing():
    # tokens sharing a remote coordinate cannot be told apart by remote RoPE alone
    L, d, theta, w_pre, w0 = 64, 16, 1e4, 16, 4
    G = oracle.group_size(L, w_pre)
    assert G == 4
    rng = np.random.default_rng(12)
    xk = rng.standard_normal((L, 1, d))
    xk[21] = xk[20]                       # same content, positions 20 and 21 share floor(k/4) = 5
    xk[25] = xk[20]                       # position 25 is in the next group
    K = _rope_np(xk, np.arange(L), theta)
    Q = _rope_np(rng.standard_normal((L, 1, d)), np.arange(L), theta)
    s = oracle.scores_row(Q[60, 0], K, 60, 0, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    assert abs(s[20] - s[21]) < 1e-6
    assert abs(s[20] - s[25]) > 1e-4
    s_loc = oracle.scores_row(Q[22, 0], K, 22, 0, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    assert abs(s_loc[20] - s_loc[21]) > 1e-4          # inside the local window they are told apart


def test_per_pair_length_is_the_same_as_truncating_the_cache():
    # decode runs: pair j with current length L_j == a separate call on the cache cut at L_j
    Ltot, H_q, H_kv, d, theta, w_pre, w0 = 50, 4, 2, 8, 1e4, 16, 3
    xq, xk, v = _raw_inputs(Ltot, H_q, H_kv, d, 13)
    Q = _rope_np(xq, np.arange(Ltot), theta)
    K = _rope_np(xk, np.arange(Ltot), theta)
    Ls = np.array([32, 33, 48, 49, 50])          # G = 2, 3, 3, 4, 4: crosses two boundaries
    rows, heads = Ls - 1, np.array([0, 1, 2, 3, 0])
    o, l = oracle.attend_rows(Q, K, v, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=theta, Ls=Ls)
    for j, L in enumerate(Ls):
        o1, l1 = oracle.attend_rows(Q[:L], K[:L], v[:L], [L - 1], [heads[j]], w_local=w0, w_pretrained=w_pre,
                                    rope_theta=theta)
        assert np.array_equal(o[j], o1[0]) and l[j] == l1[0]
    assert [oracle.group_size(int(L), w_pre) for L in Ls] == [2, 3, 3, 4, 4]


def test_bad_arguments_are_rejected():
    K = np.zeros((4, 1, 4), dtype=np.float32)
    with pytest.raises(ValueError):
        oracle.attend_rows(K, K, K, [5], [0], w_local=1, w_pretrained=2, rope_theta=1e4)
    with pytest.raises(ValueError):
        oracle.attend_rows(K, K, K, [1], [0], w_local=-1, w_pretrained=2, rope_theta=1e4)
    assert oracle.group_size(0, 5) == -1
    assert oracle.num_threads() >= 1


# ---------------------------------------------------------------- frequency-interpolation remote map (R17)
def _yarn_theta_prime(theta, d, w_pre, G, alpha=1.0, beta=32.0):
    """theta'_i of the definition, written out independently of the C code."""
    out = []
    for i in range(d // 2):
        th = theta ** (-2.0 * i / d)
        r = w_pre * th / (2.0 * math.pi)
        gam = min(1.0, max(0.0, (r - alpha) / (beta - alpha)))
        out.append(th * ((1.0 - gam) / G + gam))
    return out


def test_freq_map_from_scratch_complex_bruteforce():
    # the definition literally: remote scores = RoPE with theta' applied FROM SCRATCH to the content vectors at the TRUE
    # positions; the oracle goes the other way (stored theta-rotated operands + per-frequency correction angle)
    L, H_q, H_kv, d, theta, w_pre, w0 = 40, 4, 2, 8, 50.0, 9, 3
    xq, xk, v = _raw_inputs(L, H_q, H_kv, d, 21)
    Q = _rope_np(xq, np.arange(L), theta)
    K = _rope_np(xk, np.arange(L), theta)
    rows = np.repeat(np.arange(L), H_q)
    heads = np.tile(np.arange(H_q, dtype=np.int32), L)
    alpha, beta = 0.1, 0.9                     # a ramp that puts some of the 4 frequencies in each regime at this tiny size
    out, lse = oracle.attend_rows_freq(Q, K, v, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=theta,
                                       alpha=alpha, beta=beta)
    G = -(-L // w_pre)
    h = d // 2
    th = [theta ** (-2.0 * i / d) for i in range(h)]
    thp = _yarn_theta_prime(theta, d, w_pre, G, alpha, beta)
    assert any(abs(a - b) < 1e-15 for a, b in zip(th, thp)) and any(abs(a / G - b) < 1e-15 for a, b in zip(th, thp))
    Q32, K32, V32 = Q.astype(np.float32), K.astype(np.float32), v.astype(np.float32)
    for j, (q, hq) in enumerate(zip(rows, heads)):
        kv = hq // (H_q // H_kv)
        s = []
        for k in range(q + 1):
            acc = 0.0
            for i in range(h):
                zq = complex(Q32[q, hq, i], Q32[q, hq, i + h]) * cmath.exp(-1j * q * th[i])       # content vectors
                zk = complex(K32[k, kv, i], K32[k, kv, i + h]) * cmath.exp(-1j * k * th[i])
                f = th[i] if q - k <= w0 else thp[i]
                acc += (zq * cmath.exp(1j * q * f) * (zk * cmath.exp(1j * k * f)).conjugate()).real
            s.append(acc / math.sqrt(d))
        m = max(s)
        p = [math.exp(t - m) for t in s]
        l = sum(p)
        o = [sum(p[k] * float(V32[k, kv, c]) for k in range(q + 1)) / l for c in range(d)]
        assert np.allclose(out[j], o, atol=1e-12)
        assert abs(lse[j] - (m + math.log(l))) < 1e-12


def test_freq_map_special_cases():
    L, H_q, H_kv, d, theta, w0 = 60, 2, 1, 16, 1e4, 5
    xq, xk, v = _raw_inputs(L, H_q, H_kv, d, 22)
    Q = _rope_np(xq, np.arange(L), theta).astype(np.float32)
    K = _rope_np(xk, np.arange(L), theta).astype(np.float32)
    rows = np.repeat(np.arange(L), H_q)
    heads = np.tile(np.arange(H_q, dtype=np.int32), L)
    ctrl = oracle.attend_rows(Q, K, v, rows, heads, w_local=w0, w_pretrained=16, rope_theta=theta, mode="causal")
    # G = 1: phi = 0, the map is the identity -> the control, bit for bit (cos 0 = 1, sin 0 = 0)
    g1 = oracle.attend_rows_freq(Q, K, v, rows, heads, w_local=w0, w_pretrained=L, rope_theta=theta)
    assert np.array_equal(g1[0], ctrl[0]) and np.array_equal(g1[1], ctrl[1])
    # gamma = 1 for every frequency (ramp far below every r_i): nothing is interpolated -> the control
    hi = oracle.attend_rows_freq(Q, K, v, rows, heads, w_local=w0, w_pretrained=16, rope_theta=theta, alpha=-2e9, beta=-1e9)
    assert np.array_equal(hi[0], ctrl[0]) and np.array_equal(hi[1], ctrl[1])
    # gamma = 0 for every frequency: position interpolation x -> x / G; with every pair of x_q, x_k equal to (1, 0) the
    # remote score is the closed form sum_i cos((q - k) theta_i / G) / sqrt(d), the local one sum_i cos((q - k) theta_i)
    ones = np.zeros((L, 1, d)); ones[..., : d // 2] = 1.0
    Q1 = _rope_np(ones, np.arange(L), theta).astype(np.float32)
    K1 = _rope_np(ones, np.arange(L), theta).astype(np.float32)
    V1 = np.zeros((L, 1, d), dtype=np.float32)
    q = L - 1
    w_pre = 16
    G = -(-L // w_pre)
    o, lse = oracle.attend_rows_freq(Q1, K1, V1, [q], [0], w_local=w0, w_pretrained=w_pre, rope_theta=theta, alpha=1e30, beta=2e30)
    th = theta ** (-2.0 * np.arange(d // 2) / d)
    s = [(np.cos((q - k) * th).sum() if q - k <= w0 else np.cos((q - k) * th / G).sum()) / math.sqrt(d) for k in range(q + 1)]
    assert abs(lse[0] - math.log(sum(math.exp(t) for t in s))) < 1e-5          # fp32 rounding of the generated inputs
    # interpolation keeps RELATIVE positions: a global shift of every position by ANY c changes nothing
    # (aliasing is invariant only for c divisible by G, test_shift_invariance)
    base = oracle.attend_rows_freq(Q, K, v, rows, heads, w_local=w0, w_pretrained=16, rope_theta=theta)
    for c in (1, 7, 1000):
        sh = oracle.attend_rows_freq(Q, K, v, rows, heads, w_local=w0, w_pretrained=16, rope_theta=theta, pos_shift=c)
        assert np.abs(sh[0] - base[0]).max() < 1e-9 and np.abs(sh[1] - base[1]).max() < 1e-9
    # and it differs from aliasing and from the control on these inputs
    ali = oracle.attend_rows(Q, K, v, rows, heads, w_local=w0, w_pretrained=16, rope_theta=theta)
    assert np.abs(base[1] - ali[1]).max() > 1e-3 and np.abs(base[1] - ctrl[1]).max() > 1e-3
