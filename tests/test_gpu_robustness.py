"""GPU tests of what a parity run on one seed does not show: the margin of the default precision over many seeds and
adversarial inputs, the fallback shapes, run-to-run determinism, repeats, stream capture, concurrent host threads with
different options, and stream ordering of decode behind a kernel that writes its inputs."""
import threading

import numpy as np
import pytest
import torch

import paper_2607_07740_b200 as J
from paper_2607_07740_b200 import binding as B
from paper_2607_07740_b200 import workloads as W

from parity_util import TOL, all_pairs, check, gather, oracle_rows

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _lse_err(Q, K, V, rows, heads, **kw):
    out, lse = J.jetlong_prefill(Q, K, V, **kw)
    torch.cuda.synchronize()
    ro, rl = oracle_rows(Q, K, V, rows, heads, w_local=kw["w_local"], w_pretrained=kw["w_pretrained"], rope_theta=kw["rope_theta"])
    og, lg = gather(out, lse, rows, heads)
    eo = np.abs(og.double().cpu().numpy() - ro).max()
    el = np.abs(lg.double().cpu().numpy() - rl).max()
    return float(eo), float(el)


def _pick(L, H_q, n, seed):
    rows, heads = all_pairs(L, H_q)
    if len(rows) > n:
        sel = np.random.RandomState(seed).choice(len(rows), n, replace=False)
        rows, heads = rows[sel], heads[sel]
    return rows, heads


# ---- margin of the DEFAULT precision (selective e5m2 compensation): 32 seeds x three lengths, then adversarial inputs -------
@pytest.mark.parametrize("L,w_pre,w0", [(777, 200, 100), (4096, 1024, 128), (8320, 2048, 256)])
def test_default_precision_margin_over_seeds(L, w_pre, w0):
    worst_o = worst_l = 0.0
    for s in range(32):
        Q, K, V = W.make_qkv(L, 4, 2, 128, 1e6, "bf16", 50000 + 97 * s + L, True, DEV)
        rows, heads = _pick(L, 4, 1536, s)
        eo, el = _lse_err(Q, K, V, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=1e6)
        worst_o, worst_l = max(worst_o, eo), max(worst_l, el)
    print("default precision, L=%d, 32 seeds: worst out %.3e, worst lse %.3e" % (L, worst_o, worst_l))
    assert worst_l <= TOL[torch.bfloat16]["lse"] and worst_o <= TOL[torch.bfloat16]["out_abs"], (worst_o, worst_l)


@pytest.mark.parametrize("profile", ["switch", "q_outliers", "loud"])
def test_default_precision_on_adversarial_inputs(profile):
    """Outlier channels that change halfway through the sequence, outliers in Q only, every K channel x1.5: the
    selection works from global mean energies, these inputs are what it cannot see well."""
    worst_l = worst_o = 0.0
    for L, w_pre, w0 in ((4096, 1024, 128), (8320, 2048, 256)):
        for s in range(6):
            Q, K, V = W.make_qkv(L, 4, 2, 128, 1e6, "bf16", 61000 + 13 * s + L, True, DEV, profile=profile)
            rows, heads = _pick(L, 4, 1536, s)
            eo, el = _lse_err(Q, K, V, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=1e6)
            worst_o, worst_l = max(worst_o, eo), max(worst_l, el)
    print("default precision, profile %s: worst out %.3e, worst lse %.3e" % (profile, worst_o, worst_l))
    assert worst_l <= TOL[torch.bfloat16]["lse"] and worst_o <= TOL[torch.bfloat16]["out_abs"], (profile, worst_o, worst_l)


def test_default_precision_margin_on_config_rows():
    """The same at the sizes bench.py times: C2 and C3 sampled rows; prints the maxima so the margin is on record."""
    for c in (W.C2, W.C3):
        Q, K, V = W.make_config_inputs(c, DEV)
        G = J.jetlong_group_size(c.L, c.w_pretrained)
        rows, heads = W.sample_pairs(c.L, c.H_q, 512, c.seed() + 5, c.w_local, G)
        eo, el = _lse_err(Q, K, V, rows, heads, w_local=c.w_local, w_pretrained=c.w_pretrained, rope_theta=c.rope_theta)
        print("%s: out %.3e lse %.3e" % (c.name, eo, el))
        assert el <= 7e-4 and eo <= 2e-2, (c.name, eo, el)
        del Q, K, V


# ---- odd GQA groups and MHA run on the tcgen05 two-tile kernel too: the lone head of a group is served by one CTA pair on
# four consecutive query blocks (prefill_umma2.cu); only fp32 and head_dim 64 use the SIMT tiles --------------------------
@pytest.mark.parametrize("L,H_q,H_kv,w_pre,w0", [
    (700, 3, 1, 200, 64),          # g = 3: one head pair + one lone head; 6 query blocks (ragged 512-row block)
    (700, 7, 1, 200, 64),          # g = 7, as in 28 / 4-head models
    (700, 5, 5, 200, 64),          # MHA: every head is a lone head
    (2200, 7, 1, 512, 128),        # 18 query blocks, G = 5, longer remote phases
    (1300, 4, 4, 300, 0),          # MHA, w0 = 0 (joint local ranges with gaps), 11 query blocks
    (513, 1, 1, 128, 100),         # a single head
    (700, 6, 2, 200, 64),          # g = 3 with two KV heads
])
def test_bf16_d128_odd_group_sizes(L, H_q, H_kv, w_pre, w0):
    assert B.lib().jetlong_prefill_uses_umma(L, H_q, H_kv, 128) == 1
    Q, K, V = W.make_qkv(L, H_q, H_kv, 128, 1e6, "bf16", 4400 + H_q + L, True, DEV)
    rows, heads = all_pairs(L, H_q)
    for name, fn in (("bifocal", lambda: J.jetlong_prefill(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=1e6)),
                     ("workspace variant", lambda: J.jetlong_prefill_prerotated(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=1e6))):
        out, lse = fn()
        ro, rl = oracle_rows(Q, K, V, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=1e6)
        check(*gather(out, lse, rows, heads), ro, rl, Q.dtype, "%s g=%d/%d L=%d" % (name, H_q, H_kv, L))
    out, lse = J.jetlong_causal_prefill(Q, K, V)
    ro, rl = oracle_rows(Q, K, V, rows, heads, w_local=0, w_pretrained=1, rope_theta=1e6, mode="causal")
    check(*gather(out, lse, rows, heads), ro, rl, Q.dtype, "control g=%d/%d L=%d" % (H_q, H_kv, L))


# ---- determinism, repeats, capture, threads ---------------------------------------------------------------------------------
def test_prefill_is_bitwise_repeatable():
    L, w_pre, w0 = 8320, 2048, 256
    Q, K, V = W.make_qkv(L, 4, 2, 128, 1e6, "bf16", 31, True, DEV)
    ref = None
    for _ in range(5):
        out, lse = J.jetlong_prefill(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=1e6)
        torch.cuda.synchronize()
        if ref is None:
            ref = (out.clone(), lse.clone())
        assert torch.equal(out, ref[0]) and torch.equal(lse, ref[1])


@pytest.mark.parametrize("impl", [4, 1])
def test_prefill_repeated_200_times(impl):
    """A rare mbarrier-phase slip would show as a hang (pytest timeout) or a changed result."""
    ref = {}
    shapes = ((777, 200, 100), (1300, 300, 0), (2200, 512, 128))
    data = {s: W.make_qkv(s[0], 4, 2, 128, 1e6, "bf16", 700 + s[0], True, DEV) for s in shapes}
    ws = {s: B.alloc_workspace(B.OP_PREFILL, s[0], 4, 2, 128, B.BF16, DEV) for s in shapes}
    for it in range(200):
        for s in shapes:
            Q, K, V = data[s]
            out, lse = J.jetlong_prefill(Q, K, V, w_local=s[2], w_pretrained=s[1], rope_theta=1e6, impl=impl, workspace=ws[s])
            if it % 50 == 0 or it == 199:
                torch.cuda.synchronize()
                if s not in ref:
                    ref[s] = (out.clone(), lse.clone())
                assert torch.equal(out, ref[s][0]) and torch.equal(lse, ref[s][1]), (s, it)
    torch.cuda.synchronize()


def test_prefill_under_stream_capture():
    L, w_pre, w0 = 4096, 1024, 128
    Q, K, V = W.make_qkv(L, 4, 2, 128, 1e6, "bf16", 32, True, DEV)
    ws = B.alloc_workspace(B.OP_PREFILL, L, 4, 2, 128, B.BF16, DEV)
    out = torch.empty_like(Q)
    lse = torch.empty((4, L), dtype=torch.float32, device=DEV)
    eager_o, eager_l = J.jetlong_prefill(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=1e6)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        J.jetlong_prefill(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=1e6, out=out, lse=lse, workspace=ws)
    out.zero_(); lse.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out, eager_o) and torch.equal(lse, eager_l)
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out, eager_o) and torch.equal(lse, eager_l)


def test_two_host_threads_with_different_options():
    """Two threads, two streams, different precisions, at the same time: each gets the result of ITS options
    (nothing in the launch path is process-global; the setters are per-thread)."""
    L, w_pre, w0 = 4096, 1024, 128
    Q, K, V = W.make_qkv(L, 4, 2, 128, 1e6, "bf16", 33, True, DEV)
    want = {}
    for name, mode in (("fast", B.PRECISION_FAST), ("e5m2", B.PRECISION_COMPENSATED_E5M2)):
        o, l = J.jetlong_prefill(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=1e6, precision=mode)
        torch.cuda.synchronize()
        want[name] = (o.clone(), l.clone())
    assert not torch.equal(want["fast"][1], want["e5m2"][1])        # the two modes differ, so a mix-up is visible
    errors = []

    def worker(name, mode, use_setter):
        try:
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                if use_setter:
                    J.jetlong_set_prefill_precision(mode)           # this thread's default only
                for _ in range(20):
                    kw = {} if use_setter else {"precision": mode}
                    o, l = J.jetlong_prefill(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=1e6, **kw)
                    st.synchronize()
                    if not (torch.equal(o, want[name][0]) and torch.equal(l, want[name][1])):
                        errors.append(name)
        except Exception as e:                                       # noqa: BLE001
            errors.append("%s: %r" % (name, e))
    for use_setter in (False, True):
        ths = [threading.Thread(target=worker, args=("fast", B.PRECISION_FAST, use_setter)),
               threading.Thread(target=worker, args=("e5m2", B.PRECISION_COMPENSATED_E5M2, use_setter))]
        for t in ths:
            t.start()
        for t in ths:
            t.join()
    assert not errors, errors


# ---- decode right behind a kernel that writes its inputs (programmatic dependent launch must not read early) -----------------
@pytest.mark.parametrize("kind", ["control", "g1", "bifocal"])
def test_decode_reads_inputs_written_just_before_it(kind):
    L, H_q, H_kv, d = 6000, 32, 8, 128
    w_pre = 100000 if kind == "g1" else 2048                         # g1: L <= w_pretrained -> G = 1 -> the control path
    Qs, Kc, Vc = W.make_qkv(L, H_q, H_kv, d, 1e6, "bf16", 88, True, DEV, q_pos0=L - 1, n_q=16)
    ws = B.alloc_workspace(B.OP_DECODE, L, H_q, H_kv, d, B.BF16, DEV)
    q = torch.zeros_like(Qs[0])
    krow, vrow = Kc[L - 1].clone(), Vc[L - 1].clone()

    def call(qq):
        if kind == "control":
            return J.jetlong_causal_decode(qq, Kc, Vc, L, workspace=ws)
        return J.jetlong_decode(qq, Kc, Vc, L, w_local=512, w_pretrained=w_pre, rope_theta=1e6, workspace=ws)
    want = []
    for t in range(16):
        o, l = call(Qs[t].contiguous())
        torch.cuda.synchronize()
        want.append((o.clone(), l.clone()))
    big = torch.empty(64 << 20, dtype=torch.uint8, device=DEV)
    for rep in range(3):
        for t in range(16):
            big.fill_(rep)                                           # keeps the stream busy in front of the writers
            Kc[L - 1].zero_(); Vc[L - 1].zero_()
            q.copy_(Qs[t])                                           # the kernels that write q and KV row L-1 ...
            Kc[L - 1].copy_(krow); Vc[L - 1].copy_(vrow)
            o, l = call(q)                                           # ... immediately followed by the decode
            o, l = o.clone(), l.clone()
            torch.cuda.synchronize()
            assert torch.equal(o, want[t][0]) and torch.equal(l, want[t][1]), (kind, rep, t)


def test_table_header_is_not_trusted_when_the_body_was_overwritten():
    """A workspace whose header survived but whose table body was overwritten must be rebuilt (include/jetlong.h)."""
    L, w_pre, w0 = 3000, 512, 128
    Q, K, V = W.make_qkv(L, 4, 2, 128, 1e6, "bf16", 34, True, DEV)
    ws = B.alloc_workspace(B.OP_PREFILL, L, 4, 2, 128, B.BF16, DEV)
    o1, l1 = J.jetlong_prefill(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=1e6, workspace=ws)
    torch.cuda.synchronize()
    ws[256:].fill_(0x3c)                                             # the header stays, the tables are garbage
    o2, l2 = J.jetlong_prefill(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=1e6, workspace=ws)
    torch.cuda.synchronize()
    assert torch.equal(o1, o2) and torch.equal(l1, l2)


# ---- the host-buffer call: chunked upload / compute / download pipeline ------------------------------------------------------
@pytest.mark.parametrize("L,H_q,H_kv,d,dtype,w_pre,w0", [
    (9000, 4, 2, 128, "bf16", 2048, 256),       # 4 row chunks on the two-tile kernel, ragged last chunk
    (33000, 2, 1, 128, "bf16", 8192, 512),      # 8 chunks, an odd (lone-head) group
    (700, 4, 2, 128, "bf16", 200, 64),          # one chunk
    (1024, 4, 2, 64, "fp32", 256, 64),          # config-1 shape through the SIMT tiles
])
def test_prefill_host_pipeline(L, H_q, H_kv, d, dtype, w_pre, w0):
    theta = 1e6 if d == 128 else 1e4
    Q, K, V = W.make_qkv(L, H_q, H_kv, d, theta, dtype, 5150 + L, dtype == "bf16", DEV)
    Qh, Kh, Vh = Q.cpu().pin_memory(), K.cpu().pin_memory(), V.cpu().pin_memory()
    for _ in range(2):                                               # the second call reuses the arena
        out, lse = J.jetlong_prefill_host(Qh, Kh, Vh, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    rows, heads = _pick(L, H_q, 1024, 7)
    edge = np.array([0, 511, 512, 513, L // 2, L - 1])
    rows = np.concatenate([rows, np.repeat(edge, H_q)])
    heads = np.concatenate([heads, np.tile(np.arange(H_q, dtype=np.int32), len(edge))])
    ro, rl = oracle_rows(Q, K, V, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
    ri, hi = torch.as_tensor(rows), torch.as_tensor(heads).long()
    check(out[ri, hi], lse[hi, ri], ro, rl, Q.dtype, "host pipeline L=%d" % L)
    assert torch.isfinite(out.float()).all() and torch.isfinite(lse).all()


# ---- decode: the second-order treatment of the slow frequency pairs (DESIGN.md 5.3 SPLIT) ------------------------------
@pytest.mark.parametrize("theta,profile", [(1e6, None), (1e6, "slow_pairs"), (5e5, None), (5e5, "slow_pairs"), (4.6e5, None),
                                           (4.6e5, "slow_pairs"), (4.5e5, None)],
                         ids=["theta1e6", "theta1e6_loud", "llama3_theta", "llama3_theta_loud", "theta_at_the_bound",
                              "theta_at_the_bound_loud", "theta_below_the_bound"])
def test_decode_slow_pair_expansion_margin(theta, profile):
    """Decode rows against the oracle over seeds, lengths and group sizes (G = 2, 3, 5, 7: 128 % G == 0 and != 0, so both
    steps of the per-tile reference row occur), with the standard inputs and with the loud channels put on pairs 32 / 33,
    where the truncated third-order term is largest; rope_theta = 4.6e5 sits on the bound that admits the expansion (4.54e5),
    4.5e5 just below it (per-key rotation of all pairs, standard inputs)."""
    H_q, H_kv, d, w0 = 8, 2, 128, 256
    worst_o = worst_l = 0.0
    for L, w_pre in ((4000, 2048), (9000, 3072), (20000, 4096), (33333, 5000)):
        assert J.jetlong_group_size(L, w_pre) in (2, 3, 5, 7)
        for s in range(4):
            Q, K, V = W.make_qkv(L, H_q, H_kv, d, theta, "bf16", 71000 + 31 * s + L, profile is None, DEV,
                                 q_pos0=L - 1, n_q=1, profile=profile)
            out, lse = J.jetlong_decode(Q[0].contiguous(), K, V, L, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
            torch.cuda.synchronize()
            ro, rl = oracle_rows(Q, K, V, [L - 1] * H_q, list(range(H_q)), w_local=w0, w_pretrained=w_pre, rope_theta=theta,
                                 q_pos_rows=[0] * H_q)
            worst_o = max(worst_o, float(np.abs(out.double().cpu().numpy() - ro).max()))
            worst_l = max(worst_l, float(np.abs(lse.double().cpu().numpy() - rl).max()))
    print("decode, theta %.3g, profile %s: worst out %.3e, worst lse %.3e" % (theta, profile, worst_o, worst_l))
    assert worst_l <= TOL[torch.bfloat16]["lse"] and worst_o <= TOL[torch.bfloat16]["out_abs"], (worst_o, worst_l)


def test_coincident_loud_pairs_switch_the_selected_cross_terms_to_fp16():
    """the same frequency pairs loud in Q (x4) AND in K (x8).  With e5m2 cross terms the default precision
    measured 3.4e-3 of lse here; the selection kernel now flags such heads and the two-tile kernel keeps the SELECTED pairs'
    cross terms in fp16 (7e-4 .. 1e-3: what is left is the un-averaged noise of the pairs left out, the softmax of these rows
    is peaked).  PRECISION_COMPENSATED_F16 (every pair in fp16, per call) stays the reference point at 4e-5."""
    L, w_pre, w0, theta = 8320, 2048, 256, 1e6
    errs = {}
    for seed in (61000 + L, 61013 + L):
        Q, K, V = W.make_qkv(L, 4, 2, 128, theta, "bf16", seed, False, DEV, profile="slow_pairs")
        rows, heads = _pick(L, 4, 1024, 5)
        ro, rl = oracle_rows(Q, K, V, rows, heads, w_local=w0, w_pretrained=w_pre, rope_theta=theta)
        for name, prec in (("default", J.PRECISION_COMPENSATED), ("fp16 cross terms", J.PRECISION_COMPENSATED_F16)):
            out, lse = J.jetlong_prefill(Q, K, V, w_local=w0, w_pretrained=w_pre, rope_theta=theta, precision=prec)
            torch.cuda.synchronize()
            og, lg = gather(out, lse, rows, heads)
            assert torch.isfinite(og.float()).all() and torch.isfinite(lg).all()
            eo = float(np.abs(og.double().cpu().numpy() - ro).max())
            el = float(np.abs(lg.double().cpu().numpy() - rl).max())
            errs[name] = (max(errs.get(name, (0, 0))[0], eo), max(errs.get(name, (0, 0))[1], el))
    print("coincident loud pairs (Q x4, K x8): %s" % errs)
    assert errs["fp16 cross terms"][1] <= TOL[torch.bfloat16]["lse"] and errs["fp16 cross terms"][0] <= TOL[torch.bfloat16]["out_abs"]
    # the default: at the tolerance, not comfortably inside it (1e-3); 1.5e-3 would mean the flag or the fp16 path broke
    assert errs["default"][1] <= 1.5e-3 and errs["default"][0] <= TOL[torch.bfloat16]["out_abs"]
