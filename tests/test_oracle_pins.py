"""Pins for oracle/sekv_oracle.py (CPU only).

Each oracle function is checked against something OTHER than itself: numbers the paper prints
(tests/golden/*.txt, each with its citation), hand-worked examples, closed forms, LAPACK, torch's
dense scaled-dot-product attention, and brute force on tiny inputs -- chosen so that a dropped term,
a wrong sign / index / scale or a transposed operand fails at least one of them.
"""
from __future__ import annotations

import itertools
import math

import numpy as np
import pytest
import torch

from oracle import sekv_oracle as O
from tests.helpers import oracle_tables, read_golden, rel_l2, to_np
from workloads import get_spec, make_layer_inputs, make_layouts, make_queries


# ---------------------------------------------------------------------------------------------
# storage rounding
# ---------------------------------------------------------------------------------------------
def test_round_bf16_matches_torch():
    rng = np.random.default_rng(1)
    x = np.concatenate([rng.standard_normal(4096) * 10.0 ** rng.integers(-8, 8, 4096),
                        [0.0, -0.0, 1.0, 1.00390625, 1.0 + 2 ** -8, 1.0 + 3 * 2 ** -9, 3.3895e38]])
    ref = torch.from_numpy(x.astype(np.float32)).to(torch.bfloat16).to(torch.float32).numpy()
    got = O.round_bf16(x)
    assert np.array_equal(got.astype(np.float32), ref)
    # ties-to-even, by hand: 1 + 2^-8 is exactly between 1 and 1 + 2^-7 -> rounds to even (1.0)
    assert O.round_bf16(np.array([1.0 + 2 ** -8]))[0] == 1.0
    assert O.round_bf16(np.array([1.0 + 3 * 2 ** -8]))[0] == 1.0 + 2 ** -6


# ---------------------------------------------------------------------------------------------
# 3.1 segmentation
# ---------------------------------------------------------------------------------------------
def _golden_H(g):
    H = np.full(int(g["n"][0]), g["low_value"][0])
    H[[int(p) for p in g["high_positions"]]] = g["high_value"][0]
    return H


def test_segmentation_hand_worked_example():
    g = read_golden("segmentation_planted.txt")
    H = _golden_H(g)
    assert O.surprisal_threshold(H, g["alpha"][0]) == pytest.approx(g["threshold"][0], abs=1e-12)
    for tag, lmin, win in (("lmin4", 4, 0), ("lmin5", 5, 0), ("lmin5_w3", 5, 3)):
        seg = O.segment(H, alpha=1.0, l_min=lmin, window=win)
        assert seg.span_start.tolist() == [int(x) for x in g[f"{tag}_span_start"]], tag
        assert seg.span_len.tolist() == [int(x) for x in g[f"{tag}_span_len"]], tag
        assert seg.pool_pos.tolist() == [int(x) for x in g[f"{tag}_pool"]], tag


def test_segmentation_strict_inequality_and_population_sigma():
    # H = (0, 4): mu = 2, population sigma = 2 (exact in binary), sample sigma = 2.83.
    # alpha = 1 puts the threshold exactly at 4 with the population sigma: strict '>' => no boundary
    # (one span of 2).  A sample-sigma reading would agree there, so also check alpha = 0.9:
    # population thr = 3.8 < 4 -> token 1 is a boundary; sample thr = 4.55 -> none.
    H = np.array([0.0, 4.0])
    assert O.surprisal_threshold(H, 1.0) == 4.0
    seg = O.segment(H, alpha=1.0, l_min=1)
    assert seg.A == 0 and seg.span_len.tolist() == [2]
    seg = O.segment(H, alpha=0.9, l_min=1)
    assert seg.pool_pos.tolist() == [1] and seg.span_len.tolist() == [1]


def test_segmentation_constant_surprisal_is_one_span():
    seg = O.segment(np.full(100, 2.5), alpha=1.0, l_min=16)
    assert seg.A == 0 and seg.span_start.tolist() == [0] and seg.span_len.tolist() == [100]


@pytest.mark.parametrize("cid", [0, 1])
def test_segmentation_recovers_planted_layout_and_partitions_tokens(cid):
    spec = get_spec(cid)
    for l in make_layouts(spec):
        seg = O.segment(l.H, spec.alpha, spec.l_min, spec.window)
        assert np.array_equal(seg.span_start, l.planted_span_start)
        assert np.array_equal(seg.span_len, l.planted_span_len)
        assert np.array_equal(seg.pool_pos, l.planted_pool_pos)
        # invariants: partition of [0, n), spans disjoint/ordered/>= L_min
        assert int(seg.span_len.sum()) + seg.A == l.n
        assert (seg.span_len >= spec.l_min).all()
        assert (seg.span_start[1:] >= seg.span_start[:-1] + seg.span_len[:-1]).all()
        covered = np.zeros(l.n, dtype=int)
        covered[seg.pool_pos] += 1
        for a, ln in zip(seg.span_start, seg.span_len):
            covered[a:a + ln] += 1
        assert (covered == 1).all()


# ---------------------------------------------------------------------------------------------
# 3.2 summaries and factors
# ---------------------------------------------------------------------------------------------
def test_span_weights_and_summaries():
    rng = np.random.default_rng(2)
    n, d, dp = 37, 16, 8
    Hs = rng.uniform(0.5, 1.5, n)
    K = rng.standard_normal((n, d))
    W = rng.standard_normal((dp, d))
    w = O.span_weights(Hs)
    assert w.sum() == pytest.approx(1.0, abs=1e-14)
    assert w[3] / w[5] == pytest.approx(Hs[3] / Hs[5], rel=1e-14)            # proportional to H
    assert np.allclose(O.span_weights(np.zeros(5)), 0.2)                      # reading #6
    kbar = O.coarse_mean(w, K)
    # brute-force definition, element by element
    ref = [sum(Hs[t] / Hs.sum() * K[t, j] for t in range(n)) for j in range(d)]
    assert np.allclose(kbar, ref, atol=1e-14)
    # constant surprisal => plain mean (BASELINE.json configs[0] "summary = mean of span keys")
    assert np.allclose(O.coarse_mean(O.span_weights(np.full(n, 0.7)), K), K.mean(axis=0), atol=1e-14)
    Kb = O.routing_summary(w, K, W)
    assert np.sqrt((Kb ** 2).sum()) == pytest.approx(1.0, abs=1e-14)           # Eq. 3 normalisation
    lin = W @ kbar                                                             # linearity of Eq. 3
    assert np.allclose(Kb, lin / np.linalg.norm(lin), atol=1e-13)
    # W = I, d' = d_h  => the direction of the weighted mean key
    assert np.allclose(O.routing_summary(w, K, np.eye(d)), kbar / np.linalg.norm(kbar), atol=1e-13)
    # a transposed-operand mistake (W^T) would fail this asymmetric check:
    W2 = np.zeros((dp, d)); W2[0, 1] = 1.0
    Kb2 = O.routing_summary(w, K, W2)
    assert abs(Kb2[0]) == pytest.approx(1.0) and np.allclose(Kb2[1:], 0.0)


def test_truncated_svd_eckart_young_and_known_spectrum():
    rng = np.random.default_rng(3)
    n, d = 40, 24
    Uq, _ = np.linalg.qr(rng.standard_normal((n, d)))
    Vq, _ = np.linalg.qr(rng.standard_normal((d, d)))
    sig = np.sort(rng.uniform(0.1, 3.0, d))[::-1]
    X = (Uq * sig) @ Vq.T                                   # known singular values by construction
    for r in (1, 5, 24, 64):
        U, s, Vt = O.truncated_svd(X, r)
        R = min(n, d, r)
        assert U.shape == (n, R) and s.shape == (R,) and Vt.shape == (R, d)    # Eq. 6: R = min(|S|, d_h, R_max)
        assert np.allclose(s, sig[:R], atol=1e-12)
        Xh = O.gated_reconstruction(U, s, Vt)
        # PAPER.md L145 with binary gates: ||K - K_hat||_F^2 = sum_{i>r} sigma_i^2
        gates = np.concatenate([np.ones(R), np.zeros(d - R)])
        assert ((X - Xh) ** 2).sum() == pytest.approx(O.gated_error(gates, sig), rel=1e-9, abs=1e-18)
    # soft gates: E(m, sigma) = sum (1-m_i)^2 sigma_i^2 against the explicit residual
    U, s, Vt = O.truncated_svd(X, d)
    m = rng.uniform(0, 1, d)
    Xm = O.gated_reconstruction(U, s, Vt, gates=m)
    assert ((X - Xm) ** 2).sum() == pytest.approx(O.gated_error(m, s), rel=1e-9)
    # a rank-r matrix is reconstructed to rounding
    Xr = (Uq[:, :4] * sig[:4]) @ Vq[:, :4].T
    U, s, Vt = O.truncated_svd(Xr, 4)
    assert np.allclose(O.gated_reconstruction(U, s, Vt), Xr, atol=1e-12)
    # orientation: U is [|S|, R] (token side), Vt is [R, d_h] -- an asymmetric rank-1 case
    X1 = np.outer(np.arange(1, 6), [0.0, 2.0, 0.0])
    U, s, Vt = O.truncated_svd(X1, 1)
    assert abs(Vt[0, 1]) == pytest.approx(1.0) and abs(U[4, 0]) > abs(U[0, 0])


def test_storage_count_and_byte_accounting_match_paper():
    g = read_golden("paper_appendix_d.txt")
    L, hk, d, b = (int(g[k][0]) for k in ("fullkv_L", "fullkv_H_kv", "fullkv_d_h", "fullkv_b"))
    assert O.fullkv_bytes(L, hk, d, 1, b) == g["fullkv_per_token_KB"][0] * 1024          # 192 KB / token
    assert O.fullkv_bytes(L, hk, d, 128 * 1024, b) == g["fullkv_128k_GB"][0] * 2 ** 30  # 24 GB at 128K
    p = O.routing_parameters(int(g["route_L"][0]), int(g["route_H"][0]), int(g["route_d_route"][0]),
                             int(g["route_d_h"][0]))
    assert round(p / 1e6, 2) == g["route_params_millions"][0]                            # ~4.19M
    assert int(g["route_L"][0]) * int(g["route_H"][0]) == g["route_thresholds"][0]
    assert round(100 * (1 - g["mem_sekv_128k_GB"][0] / g["mem_fullkv_128k_GB"][0]), 1) == g["mem_reduction_percent"][0]
    # r(|S| + d_h + 1) values; Eq. 18 = 2 L H_kv r(|S|+d_h+1) b; Eq. 20 sums Eq. 18
    assert O.sekv_cpu_span_values(16, 100, 128) == 16 * 229
    assert O.sekv_cpu_span_bytes(32, 8, 16, 100, 128, 2) == 2 * 32 * 8 * 16 * 229 * 2
    assert O.transfer_bytes(32, 8, 16, [100, 50], 128, 2) == 2 * 32 * 8 * 16 * (229 + 179) * 2
    # Eq. 17 with d' << d_h is far below Eq. 16 (a + w << n)
    assert O.sekv_gpu_bytes(48, 8, 40, 128, 32, 3745, 512, 936, 2) < 0.05 * O.fullkv_bytes(48, 8, 128, 131072, 2)
    assert O.sekv_gpu_bytes(1, 1, 1, 128, 32, 10, 2, 5, 2) == 2 * 128 * 12 * 2 + 2 * 32 * 5 * 2


def test_build_tables_dense_matches_components_and_rounding():
    spec = get_spec(0).with_(contexts=(700,))
    lay = make_layouts(spec)
    li = make_layer_inputs(spec, lay, 0, dense=True)
    T = oracle_tables(spec, lay, li, 0, mode="dense", r_max=8)
    K = to_np(li.K)
    l = lay[0]
    assert np.array_equal(T.full_K[0], K[0, l.planted_pool_pos])
    s = 2
    a, ln = int(T.seg.span_start[s]), int(T.seg.span_len[s])
    w = l.H[a:a + ln].astype(np.float64); w = w / w.sum()
    assert np.allclose(T.mean_K[0, s], (w[:, None] * K[0, a:a + ln]).sum(0), atol=1e-6)
    # stored factors reconstruct the (rank 8 + rounding noise) span to fp32 accuracy
    f = T.factors[0][s]
    assert f.UK.shape == (ln, 8) and f.VtK.shape == (8, 128)
    assert rel_l2(O.gated_reconstruction(f.UK, f.sK, f.VtK), K[0, a:a + ln]) < 1e-5
    # every query head of the group gets its own summary from its own W
    W = to_np(li.W)
    for h in range(4):
        ref = W[h] @ (w @ K[0, a:a + ln]); ref /= np.linalg.norm(ref)
        assert np.allclose(T.route_K[h, s], ref, atol=1e-6)


def test_build_tables_prefactored_defines_span_keys_as_products():
    spec = get_spec(1).with_(contexts=(3000,), n_q_heads=4, n_kv_heads=2)
    lay = make_layouts(spec)
    li = make_layer_inputs(spec, lay, 0)
    T = oracle_tables(spec, lay, li, 0)
    s, g = 1, 1
    a, ln = int(T.seg.span_start[s]), int(T.seg.span_len[s])
    Ks = (to_np(li.tokUK[g, a:a + ln]) * to_np(li.SK[g, s])) @ to_np(li.VtK[g, s])
    w = lay[0].H[a:a + ln].astype(np.float64); w /= w.sum()
    assert np.array_equal(T.mean_K[g, s], O.round_bf16(w @ Ks))
    assert T.factors[g][s].UV.shape == (ln, 16)
    # stored summaries are bf16 values
    assert np.array_equal(T.route_K, O.round_bf16(T.route_K))


# ---------------------------------------------------------------------------------------------
# 3.3 routing
# ---------------------------------------------------------------------------------------------
def _brute_topk(scores, k):
    """Independent selection: repeatedly take the max, lowest index first among equals."""
    left = list(range(len(scores)))
    out = []
    while left and (k < 0 or len(out) < k):
        best = left[0]
        for i in left[1:]:
            if scores[i] > scores[best]:
                best = i
        out.append(best)
        left.remove(best)
    return out


def test_sigmoid_size_prior_closed_form():
    # sig(x + ln n) = n e^x / (1 + n e^x)   (Eq. 5 with the log|S| prior)
    for x, n in itertools.product([-3.0, -0.2, 0.0, 1.7], [1, 16, 137, 256]):
        assert O.sigmoid(x + math.log(n)) == pytest.approx(n * math.exp(x) / (1 + n * math.exp(x)), rel=1e-13)


def test_route_against_elementwise_definition_and_brute_force():
    rng = np.random.default_rng(5)
    hq, hk, d, dp, m = 6, 2, 16, 4, 23
    W = rng.standard_normal((hq, dp, d))
    q = rng.standard_normal((hq, d))
    Kb = rng.standard_normal((hq, m, dp)); Kb /= np.linalg.norm(Kb, axis=-1, keepdims=True)
    lens = rng.integers(16, 257, m)
    R = O.route(q, W, Kb, lens, hk, k=5)
    for h, s in [(0, 0), (3, 7), (5, 22)]:
        qp = [sum(W[h, j, c] * q[h, c] for c in range(d)) for j in range(dp)]               # Eq. 4
        x = sum(qp[j] * Kb[h, s, j] for j in range(dp)) / math.sqrt(dp) + math.log(lens[s])  # Eq. 5
        assert R.logit[h, s] == pytest.approx(x, rel=1e-12)
        assert R.alpha[h, s] == pytest.approx(1 / (1 + math.exp(-x)), rel=1e-12)
    # order by alpha == order by logit where alpha has not saturated
    assert np.array_equal(np.argsort(-R.logit[0], kind="stable"), np.argsort(-R.alpha[0], kind="stable"))
    G = hq // hk
    for g in range(hk):
        X = R.logit[g * G:(g + 1) * G].max(axis=0)
        assert np.array_equal(R.group_logit[g], X)
        assert R.ids[g].tolist() == _brute_topk(X.tolist(), 5)
    assert [len(i) for i in O.route(q, W, Kb, lens, hk, k=0).ids] == [0, 0]
    allr = O.route(q, W, Kb, lens, hk, k=-1)
    assert sorted(allr.ids[0].tolist()) == list(range(m))
    assert O.route(q, W, Kb, lens, hk, k=1000).ids[1].tolist() == allr.ids[1].tolist()
    # G = 1 reduces to the paper's per-query-head rule exactly
    R1 = O.route(q, W, Kb, lens, hq, k=3)
    for h in range(hq):
        assert R1.ids[h].tolist() == _brute_topk(R1.logit[h].tolist(), 3)


def test_route_ties_go_to_lower_id_and_threshold_rule():
    rng = np.random.default_rng(6)
    hq, hk, d, dp, m = 2, 1, 8, 4, 9
    W = rng.standard_normal((hq, dp, d)); q = rng.standard_normal((hq, d))
    Kb = rng.standard_normal((hq, m, dp)); Kb /= np.linalg.norm(Kb, axis=-1, keepdims=True)
    lens = np.full(m, 32)
    Kb[:, 6] = Kb[:, 2]                      # exact duplicate span: exact tie in every head
    R = O.route(q, W, Kb, lens, hk, k=-1)
    order = R.ids[0].tolist()
    assert order.index(2) + 1 == order.index(6)
    # Eq. 9: z = 1[alpha > tau]; eligible if ANY head of the group passes; cap keeps the best
    tau = np.array([np.sort(R.alpha[0])[-3] - 1e-12, 2.0])      # head 0 passes its top 3, head 1 none
    Rt = O.route(q, W, Kb, lens, hk, k=-1, tau=tau)
    assert set(Rt.ids[0].tolist()) == set(np.argsort(-R.alpha[0])[:3].tolist())
    Rt2 = O.route(q, W, Kb, lens, hk, k=2, tau=tau)
    assert Rt2.ids[0].tolist() == Rt.ids[0].tolist()[:2]
    # strict '>' in Eq. 9: tau equal to the best alpha selects nothing for that head
    tau_eq = np.array([R.alpha[0].max(), 2.0])
    assert len(O.route(q, W, Kb, lens, hk, k=-1, tau=tau_eq).ids[0]) == 0


# ---------------------------------------------------------------------------------------------
# 3.3 mixed-resolution attention
# ---------------------------------------------------------------------------------------------
def _sdpa(q, K, V, bias=None):
    """torch's dense scaled-dot-product attention (library routine), fp64 on CPU."""
    qt = torch.from_numpy(np.asarray(q, dtype=np.float64))[None, None, None, :]
    Kt = torch.from_numpy(np.asarray(K, dtype=np.float64))[None, None]
    Vt = torch.from_numpy(np.asarray(V, dtype=np.float64))[None, None]
    mask = None if bias is None else torch.from_numpy(np.asarray(bias, dtype=np.float64))[None, None, None, :]
    return torch.nn.functional.scaled_dot_product_attention(qt, Kt, Vt, attn_mask=mask)[0, 0, 0].numpy()


def _tiny_tables(seed=7, n=400, hq=4, hk=2, d=16, dp=4, r_max=16, l_min=4, dtype="f32"):
    rng = np.random.default_rng(seed)
    H = rng.uniform(0.5, 1.5, n)
    H[rng.choice(n, size=n // 25, replace=False)] = 9.0
    K = rng.standard_normal((hk, n, d)); V = rng.standard_normal((hk, n, d))
    W = rng.standard_normal((hq, dp, d))
    T = O.build_tables(H, K, V, W, alpha=1.0, l_min=l_min, r_max=r_max, dtype=dtype)
    return H, K, V, W, T, rng


def test_attention_closed_form_example():
    g = read_golden("attention_closed_form.txt")
    d = 4
    seg = O.Segmentation(n=9, pool_pos=np.array([0]), span_start=np.array([1, 4]), span_len=np.array([3, 5]))
    fA = O.SpanFactors(UK=np.ones((3, 1)) / math.sqrt(3), sK=np.array([0.0]), VtK=np.array([[1.0, 0, 0, 0]]),
                       UV=np.ones((3, 1)) / math.sqrt(3), sV=np.array([math.sqrt(3)]), VtV=np.array([[0, 1.0, 0, 0]]))
    fB = O.SpanFactors(UK=np.zeros((5, 1)), sK=np.zeros(1), VtK=np.zeros((1, 4)), UV=np.zeros((5, 1)),
                       sV=np.zeros(1), VtV=np.zeros((1, 4)))
    T = O.Tables(n_q_heads=1, n_kv_heads=1, head_dim=d, route_dim=2, seg=seg,
                 full_K=np.array([[[math.log(2), 0, 0, 0]]]), full_V=np.array([[[1.0, 0, 0, 0]]]),
                 mean_K=np.array([[[0.0, 0, 0, 0], [math.log(4), 0, 0, 0]]]),
                 mean_V=np.array([[[0, 1.0, 0, 0], [0, 0, 1.0, 0]]]),
                 route_K=np.zeros((1, 2, 2)), W=np.zeros((1, 2, 4)), factors=[[fA, fB]])
    q = np.array([g["q"]])
    out, lse = O.decode_attn(q, T, [[]])
    assert np.allclose(out[0], g["out_none_zoomed"], atol=1e-14)
    assert math.exp(lse[0]) == pytest.approx(g["lse_none_zoomed_exp"][0], rel=1e-13)
    out2, lse2 = O.decode_attn(q, T, [[0]])
    assert np.allclose(out2[0], g["out_A_zoomed"], atol=1e-14) and lse2[0] == pytest.approx(lse[0], rel=1e-13)


def test_full_rank_all_zoomed_equals_dense_attention():
    H, K, V, W, T, rng = _tiny_tables(r_max=16)          # r_max = d_h = 16: full rank
    q = rng.standard_normal((4, 16))
    out, lse = O.decode_attn(q, T, [list(range(T.seg.m))] * 2)
    for h in range(4):
        gk = h // 2
        assert np.allclose(out[h], _sdpa(q[h], K[gk], V[gk]), rtol=0, atol=1e-6)
        logits = K[gk] @ q[h] / 4.0
        # factors are stored rounded to fp32 here, hence 1e-7 and not 1e-12
        assert lse[h] == pytest.approx(np.log(np.exp(logits - logits.max()).sum()) + logits.max(), rel=1e-7)


def test_nothing_zoomed_attends_pool_and_coarse_entries_only():
    H, K, V, W, T, rng = _tiny_tables(r_max=4)
    q = rng.standard_normal((4, 16))
    out, _ = O.decode_attn(q, T, [[], []])
    for h in range(4):
        gk = h // 2
        keys = np.concatenate([T.full_K[gk], T.mean_K[gk]])
        vals = np.concatenate([T.full_V[gk], T.mean_V[gk]])
        bias = np.concatenate([np.zeros(T.seg.A), np.log(T.seg.span_len)])
        assert np.allclose(out[h], _sdpa(q[h], keys, vals, bias), atol=1e-10)


def test_partial_zoom_against_sdpa_over_explicit_entry_list():
    H, K, V, W, T, rng = _tiny_tables(r_max=3)
    q = rng.standard_normal((4, 16))
    zoom = [[1, 4], [0]]
    out, _ = O.decode_attn(q, T, zoom)
    for h in range(4):
        gk = h // 2
        keys, vals, bias = [T.full_K[gk]], [T.full_V[gk]], [np.zeros(T.seg.A)]
        for s in range(T.seg.m):
            if s in zoom[gk]:
                f = T.factors[gk][s]
                keys.append((f.UK * f.sK) @ f.VtK); vals.append((f.UV * f.sV) @ f.VtV)   # Eq. 8 as matmuls
                bias.append(np.zeros(f.UK.shape[0]))
            else:
                keys.append(T.mean_K[gk, s][None]); vals.append(T.mean_V[gk, s][None])
                bias.append([math.log(T.seg.span_len[s])])
        assert np.allclose(out[h], _sdpa(q[h], np.concatenate(keys), np.concatenate(vals),
                                         np.concatenate(bias)), atol=1e-10)


def test_span_permutation_changes_nothing():
    H, K, V, W, T, rng = _tiny_tables(r_max=5)
    q = rng.standard_normal((4, 16))
    zoom = [[2, 5, 0], [3]]
    out, lse = O.decode_attn(q, T, zoom)
    perm = rng.permutation(T.seg.m)                     # new index j holds old span perm[j]
    inv = np.argsort(perm)
    seg2 = O.Segmentation(n=T.seg.n, pool_pos=T.seg.pool_pos, span_start=T.seg.span_start[perm],
                          span_len=T.seg.span_len[perm])
    T2 = O.Tables(n_q_heads=4, n_kv_heads=2, head_dim=16, route_dim=4, seg=seg2, full_K=T.full_K,
                  full_V=T.full_V, mean_K=T.mean_K[:, perm], mean_V=T.mean_V[:, perm],
                  route_K=T.route_K[:, perm], W=T.W,
                  factors=[[T.factors[g][p] for p in perm] for g in range(2)])
    out2, lse2 = O.decode_attn(q, T2, [[int(inv[s]) for s in z] for z in zoom])
    assert np.allclose(out, out2, atol=1e-12) and np.allclose(lse, lse2, atol=1e-12)
    # routing scores permute with the spans
    R = O.route(q, W, T.route_K, T.seg.span_len, 2, k=4)
    R2 = O.route(q, W, T2.route_K, seg2.span_len, 2, k=4)
    assert [[int(perm[j]) for j in ids] for ids in R2.ids] == [ids.tolist() for ids in R.ids]


def test_identical_token_span_same_zoomed_or_not_and_single_token_span():
    rng = np.random.default_rng(11)
    d, n = 16, 60
    H = np.full(n, 1.0); H[[20, 41]] = 9.0
    K = rng.standard_normal((1, n, d)); V = rng.standard_normal((1, n, d))
    K[0, 0:20] = K[0, 0]; V[0, 0:20] = V[0, 0]          # span 0: 20 identical tokens
    W = rng.standard_normal((1, 4, d))
    T = O.build_tables(H, K, V, W, l_min=1, r_max=4, dtype="f32")
    q = rng.standard_normal((1, d))
    o0, l0 = O.decode_attn(q, T, [[]])
    o1, l1 = O.decode_attn(q, T, [[0]])
    assert np.allclose(o0, o1, atol=1e-6) and np.allclose(l0, l1, atol=1e-6)   # +ln|S| identity (L119)
    # |S| = 1: the coarse entry is the token itself (ln 1 = 0)
    H2 = np.full(5, 1.0); H2[[1, 3]] = 9.0
    T2 = O.build_tables(H2, K[:, :5], V[:, :5], W, l_min=1, r_max=4, dtype="f32")
    assert T2.seg.span_len.tolist() == [1, 1, 1]
    assert np.allclose(O.decode_attn(q, T2, [[]])[0][0], _sdpa(q[0], K[0, :5], V[0, :5]), atol=1e-6)


def test_factored_form_equals_materialised_and_split_merge_and_shift():
    H, K, V, W, T, rng = _tiny_tables(r_max=6)
    q = rng.standard_normal((4, 16))
    f = T.factors[1][2]
    qh = q[3]
    # logits = (U Sigma)(V^T q) == (U Sigma V^T) q   (BASELINE.json north_star)
    assert np.allclose((f.UK * f.sK) @ (f.VtK @ qh), O.gated_reconstruction(f.UK, f.sK, f.VtK) @ qh, atol=1e-12)
    zoom = [[1], [2, 3]]
    out, lse = O.decode_attn(q, T, zoom)
    for h in range(4):
        logits, values = O.mixed_entries(q[h], h // 2, T, zoom[h // 2])
        cuts = [0, 7, 7, len(logits) // 2, len(logits)]       # includes an empty part
        parts = [O.softmax_attend(logits[a:b], values[a:b]) for a, b in zip(cuts[:-1], cuts[1:])]
        o, l = O.merge_partials(parts)
        assert np.allclose(o, out[h], atol=1e-12) and l == pytest.approx(lse[h], rel=1e-12)
        # weights sum to one: constant values give that constant; shifting logits changes nothing
        oc, _ = O.softmax_attend(logits, np.full_like(values, 3.25))
        assert np.allclose(oc, 3.25, atol=1e-12)
        os_, ls = O.softmax_attend(logits + 5.0, values)
        assert np.allclose(os_, out[h], atol=1e-12) and ls == pytest.approx(lse[h] + 5.0, rel=1e-12)
        # convex hull
        assert (out[h] <= values.max(axis=0) + 1e-12).all() and (out[h] >= values.min(axis=0) - 1e-12).all()


def test_oracle_on_config0_generator_is_finite_and_consistent():
    spec = get_spec(0)
    lay = make_layouts(spec)
    li = make_layer_inputs(spec, lay, 0)
    T = oracle_tables(spec, lay, li, 0)
    q = to_np(make_queries(spec, 0))[0, 0]
    R = O.route(q, T.W, T.route_K, T.seg.span_len, spec.n_kv_heads, spec.top_k)
    assert len(R.ids[0]) == 4
    out, lse = O.decode_attn(q, T, R.ids)
    assert np.isfinite(out).all() and np.isfinite(lse).all()
    # exact-rank generator + all zoomed == dense attention over K = U S V^T and the anchors
    l = lay[0]
    K = np.zeros((l.n, 128)); V = np.zeros((l.n, 128))
    K[l.planted_pool_pos] = T.full_K[0]; V[l.planted_pool_pos] = T.full_V[0]
    for s in range(T.seg.m):
        a, ln = int(T.seg.span_start[s]), int(T.seg.span_len[s])
        f = T.factors[0][s]
        K[a:a + ln] = (f.UK * f.sK) @ f.VtK; V[a:a + ln] = (f.UV * f.sV) @ f.VtV
    out_all, _ = O.decode_attn(q, T, [list(range(T.seg.m))])
    for h in range(4):
        assert np.allclose(out_all[h], _sdpa(q[h], K, V), atol=1e-12)
