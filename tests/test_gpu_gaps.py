"""GPU parity of the paper-defined paths that the seeded configs alone do not reach:
Eq. 9's threshold rule, exact ties at the top-k cut (ties to the lower span id, position by position),
needle attention where an expanded span's coarse entry would dominate the softmax, the local window of Eq. 17,
the config-3 batch sweep and the config-4 rank sweep, deterministic CUDA-graph replay, and the report of which
kernels a batch runs on.  Every comparison is against the oracle on the library's exported tables."""
from __future__ import annotations

import numpy as np
import pytest
import torch

from oracle import sekv_oracle as O
from tests.gpu_common import TOL_BF16, compare_attn, compare_route, tables_from_export
from tests.helpers import check_ids, oracle_tables, rel_l2, to_np
from workloads import get_spec, make_layer_inputs, make_layouts, make_queries, next_queries_ar1

pytestmark = pytest.mark.gpu


def _engine(spec, lay, li=None, **kw):
    from paper_2606_31145_b200 import engine as E
    return E.create_engine(spec, lay, layer_inputs=None if li is None else [li], **kw)


def _tables(eng, spec, layer=0, factor_seqs=None):
    """Exported tables of every sequence; factors only for `factor_seqs` (None = all)."""
    from paper_2606_31145_b200.export import export_tables
    out = []
    for b in range(eng.n_seqs):
        wf = factor_seqs is None or b in factor_seqs
        out.append(tables_from_export(export_tables(eng, layer, b, wf), spec.n_q_heads, spec.n_kv_heads, spec.route_dim))
    return out


def _needle_q(T, target, scale=40.0):
    """q with W q = scale * K_bar[h, target[g]] (least squares through pinv(W)) for every query head."""
    G = T.n_q_heads // T.n_kv_heads
    q = np.zeros((1, T.n_q_heads, 128))
    for h in range(T.n_q_heads):
        q[0, h] = np.linalg.pinv(T.W[h]) @ (scale * T.route_K[h, target[h // G]])
    return torch.from_numpy(q).to(torch.bfloat16).cuda()


# ---------------------------------------------------------------------------------------------------
# (a) Eq. 9: alpha_tilde > tau, per query head, with and without the cap
# ---------------------------------------------------------------------------------------------------
def _safe_tau(alpha_h: np.ndarray, quantile: float) -> float:
    """A threshold near the given quantile of one head's alpha values that no value comes closer to than 1e-5
    (the GPU evaluates the sigmoid in fp32, the oracle in fp64: both must take the same decision)."""
    a = np.sort(alpha_h)
    i = int(quantile * (len(a) - 1))
    for d in range(len(a)):
        for j in (i + d, i - d):
            if 0 <= j < len(a) - 1 and a[j + 1] - a[j] > 4e-5:
                return float(0.5 * (a[j] + a[j + 1]))
    raise AssertionError("no gap between alpha values")


@pytest.mark.parametrize("impl", [0, 1])
def test_route_threshold_rule_eq9(impl):
    spec = get_spec(1).sharp().with_(contexts=(20000,))
    lay = make_layouts(spec)
    li = make_layer_inputs(spec, lay, 0)
    eng = _engine(spec, lay, li, impl=impl, k_cap=160, cache_ways=176)
    fused, why = eng.sekv_get_path()
    assert fused == (impl == 0), why
    tabs = _tables(eng, spec, factor_seqs=())
    T = tabs[0]
    q = make_queries(spec, 0, "cuda")[0]
    R0 = O.route(to_np(q)[0], T.W, T.route_K, T.seg.span_len, spec.n_kv_heads, -1)
    some = [_safe_tau(R0.alpha[h], 0.55 + 0.01 * (h % 9)) for h in range(spec.n_q_heads)]
    none = [1.0] * spec.n_q_heads
    allp = [0.0] * spec.n_q_heads
    mixed = [some[h] if h % 8 < 4 else 1.0 for h in range(spec.n_q_heads)]        # heads 4..7 of a group pair never pass
    for tau, k in ((some, -1), (some, 4), (some, 16), (none, 16), (allp, 16), (mixed, -1), (mixed, 8)):
        _, count, refs = compare_route(eng, 0, q, k, tabs, tau=tau)
        n_ref = [len(r) for r in refs[0].ids]
        if tau is none:
            assert n_ref == [0] * spec.n_kv_heads
        if tau is allp:
            assert n_ref == [16] * spec.n_kv_heads
        if tau is some and k == -1:
            assert all(0 < n < T.seg.m for n in n_ref), n_ref                       # some pass, some do not
    eng.close()


def test_step_with_threshold_and_cap():
    """sekv_decode_step with tau: every layer's zoom sets and outputs against the oracle (tau + cap, L123)."""
    from paper_2606_31145_b200.export import export_tables
    spec = get_spec(1).sharp().with_(n_layers=2, contexts=(16000,))
    lay = make_layouts(spec)
    eng = _engine(spec, lay, prefetch=4)
    assert eng.sekv_get_path()[0]
    L, Hq, Hkv = spec.n_layers, spec.n_q_heads, spec.n_kv_heads
    tabs = [[tables_from_export(export_tables(eng, l, 0), Hq, Hkv, spec.route_dim)] for l in range(L)]
    q = make_queries(spec, 0, "cuda")
    qn = to_np(q)
    tau = np.zeros((L, Hq))
    for l in range(L):
        T = tabs[l][0]
        R0 = O.route(qn[l, 0], T.W, T.route_K, T.seg.span_len, Hkv, -1)
        for h in range(Hq):
            tau[l, h] = _safe_tau(R0.alpha[h], 0.93 + 0.005 * (h % 8))              # ~5% of the spans pass per head
    tau_dev = torch.tensor(tau, dtype=torch.float32, device="cuda")
    out = torch.zeros((L, 1, Hq, 128), dtype=eng.out_dtype, device="cuda")
    lse = torch.zeros((L, 1, Hq), dtype=torch.float32, device="cuda")
    for step in range(2):
        eng.sekv_decode_step(q, spec.top_k, out, tau=tau_dev, lse=lse)
        torch.cuda.synchronize()
        out_h = out.float().cpu().numpy().astype(np.float64)
        for l in range(L):
            T = tabs[l][0]
            ids, count = eng.sekv_last_zoom_ids(l)
            torch.cuda.synchronize()
            R = O.route(qn[l, 0], T.W, T.route_K, T.seg.span_len, Hkv, spec.top_k, tau=tau[l])
            zoom = []
            for g in range(Hkv):
                c = int(count[0, g])
                assert c == len(R.ids[g])
                check_ids(ids[0, g, :c].cpu().numpy(), R.ids[g], R.group_logit[g])
                zoom.append([int(x) for x in ids[0, g, :c].cpu().numpy()])
            ref, _ = O.decode_attn(qn[l, 0], T, zoom)
            assert rel_l2(out_h[l, 0], ref) <= TOL_BF16["rel_l2"]
            assert np.abs(out_h[l, 0] - ref).max() <= TOL_BF16["max_abs"]
    eng.close()


# ---------------------------------------------------------------------------------------------------
# (b) exact ties at the cut: the lower span id wins, position by position (gap = 0)
# ---------------------------------------------------------------------------------------------------
def _duplicate_routing_rows(eng, layer, src, dst):
    """Make span `dst` of sequence 0 a bit-exact routing duplicate of span `src` (every query head's row)."""
    lay = eng.sekv_get_layout()
    dp, es = eng.cfg.route_dim, eng.esize
    row = dp * es
    for h in range(eng.cfg.n_q_heads):
        base = lay.route + layer * lay.route_layer_stride + h * lay.route_head_stride
        eng.dev_arena[base + dst * row: base + (dst + 1) * row] = eng.dev_arena[base + src * row: base + (src + 1) * row].clone()
    torch.cuda.synchronize()


@pytest.mark.parametrize("impl", [0, 1])
def test_exact_ties_go_to_the_lower_span_id(impl):
    spec = get_spec(1).sharp().with_(contexts=(24000,))
    lay = make_layouts(spec)
    li = make_layer_inputs(spec, lay, 0)
    eng = _engine(spec, lay, li, impl=impl)
    lens = lay[0].planted_span_len
    # three spans of equal length (equal ln|S|): s1 < s2 < s3
    trip = None
    for v in np.unique(lens):
        idx = np.nonzero(lens == v)[0]
        if len(idx) >= 3:
            trip = [int(x) for x in idx[:3]]
            break
    assert trip is not None
    s1, s2, s3 = trip
    _duplicate_routing_rows(eng, 0, s1, s2)
    _duplicate_routing_rows(eng, 0, s1, s3)
    tabs = _tables(eng, spec, factor_seqs=())
    T = tabs[0]
    assert np.array_equal(T.route_K[:, s1], T.route_K[:, s2]) and np.array_equal(T.route_K[:, s1], T.route_K[:, s3])
    q = _needle_q(T, [s1] * spec.n_kv_heads)
    qn = to_np(q)
    for k in (1, 2, 3, 4):
        R = O.route(qn[0], T.W, T.route_K, T.seg.span_len, spec.n_kv_heads, k)
        for g in range(spec.n_kv_heads):                      # the oracle's own tie rule, by construction
            assert R.group_logit[g][s1] == R.group_logit[g][s2] == R.group_logit[g][s3]
            assert list(R.ids[g][:min(k, 3)]) == trip[:min(k, 3)]
        # score outputs requested (general path) and not requested (tensor-core path of the fused kernel)
        ids_a, count_a, _ = compare_route(eng, 0, q, k, tabs)
        ids_b, count_b = eng.sekv_route(0, q, k)
        torch.cuda.synchronize()
        for ids, count in ((ids_a, count_a), (ids_b, count_b)):
            for g in range(spec.n_kv_heads):
                c = int(count[0, g])
                assert c == k
                check_ids(ids[0, g, :c].cpu().numpy(), R.ids[g], R.group_logit[g], gap=0.0)
    eng.close()


# ---------------------------------------------------------------------------------------------------
# (c) needle attention: the expanded span's coarse entry would hold 90% ... 1 - 1e-6 of the stage-1 mass
# ---------------------------------------------------------------------------------------------------
def _stage1_fraction(T, g, s, qh):
    """Share of span s's coarse entry in the softmax mass of ALL stage-1 entries (pool + every coarse entry)."""
    scale = 1.0 / np.sqrt(128.0)
    lp = (T.full_K[g] @ qh) * scale
    lc = (T.mean_K[g] @ qh) * scale + np.log(T.seg.span_len.astype(np.float64))
    mx = max(lp.max(), lc.max())
    tot = np.exp(lp - mx).sum() + np.exp(lc - mx).sum()
    return float(np.exp(lc[s] - mx) / tot)


@pytest.mark.parametrize("impl", [0, 1])
def test_needle_attention_dominant_coarse_entry_of_an_expanded_span(impl):
    """Dense build with r_max = 8.  One span s per kv head is rewritten before the build as K_t = a u + E_t, where E has
    16 equal singular values (60) in directions orthogonal to the unit vector u: the truncated SVD keeps 8 directions
    of E and drops u (singular value a sqrt|S| < 60), so k_bar_s ~ a u while the reconstructed tokens have no u
    component.  With q = c u the coarse entry of s holds 90% ... 1 - 1e-6 of the stage-1 mass and its tokens almost
    none.  PAPER.md L121: the expanded span's coarse entry is replaced by its tokens -- an implementation that adds it
    and takes it out again loses the answer to cancellation here."""
    spec = get_spec(1).with_(contexts=(2500,))
    lay = make_layouts(spec)
    li = make_layer_inputs(spec, lay, 0, dense=True)
    G, Hkv, a = spec.group, spec.n_kv_heads, 3.0
    rng = np.random.Generator(np.random.PCG64(spec.seed ^ 0xBEEF))
    target, us = [], []
    K = li.K.clone()
    long_spans = [int(i) for i in np.nonzero(lay[0].planted_span_len >= 40)[0]]
    assert len(long_spans) >= Hkv
    for g in range(Hkv):
        s = long_spans[(3 * g + 1) % len(long_spans)]
        st, ln = int(lay[0].planted_span_start[s]), int(lay[0].planted_span_len[s])
        Vd, _ = np.linalg.qr(rng.standard_normal((128, 17)))
        u, V16 = Vd[:, 0], Vd[:, 1:]
        # left factors of E orthogonal to the all-ones direction (the left singular vector of the a u term): the SVD of
        # the span is then exactly {a sqrt|S|: (1/sqrt|S|, u)} + {60 x 16: (U16, V16)}
        Ud, _ = np.linalg.qr(np.concatenate([np.ones((ln, 1)), rng.standard_normal((ln, 16))], axis=1))
        U16 = Ud[:, 1:]
        rows = a * u[None, :] + (U16 * 60.0) @ V16.T
        K[g, st:st + ln] = torch.from_numpy(rows).to(K.dtype)
        target.append(s); us.append(u)
    li.K = K
    eng = _engine(spec, lay, li, mode="dense", r_max=8, impl=impl)
    assert eng.sekv_get_path()[0] == (impl == 0)
    tabs = _tables(eng, spec)
    T = tabs[0]
    fractions = [0.9, 0.999, 1 - 1e-5, 1 - 1e-6]
    assert G == len(fractions)
    q = np.zeros((1, spec.n_q_heads, 128))
    for g in range(Hkv):
        s, u = target[g], us[g]
        f = T.factors[g][s]
        assert f.sK.shape[0] == 8 and f.sK.min() > 40.0                             # the kept components are E's
        assert np.abs(f.VtK @ u).max() < 0.05 and (T.mean_K[g, s] @ u) > 0.8 * a    # u was dropped; k_bar_s ~ a u
        for i, frac in enumerate(fractions):
            lo, hi = 0.0, 2000.0
            for _ in range(60):                                # bisection on c with the bf16-rounded query
                c = 0.5 * (lo + hi)
                if _stage1_fraction(T, g, s, O.round_bf16(c * u)) < frac:
                    lo = c
                else:
                    hi = c
            q[0, g * G + i] = O.round_bf16(hi * u)
            got = _stage1_fraction(T, g, s, q[0, g * G + i])
            assert got >= frac and (1 - got) > 0.2 * (1 - frac), (got, frac)
    qd = torch.from_numpy(q).to(torch.bfloat16).cuda()
    assert np.array_equal(to_np(qd), q)
    ids = torch.full((1, Hkv, max(eng.cfg.k_cap, 1)), -1, dtype=torch.int32, device="cuda")
    count = torch.zeros((1, Hkv), dtype=torch.int32, device="cuda")
    for g in range(Hkv):
        ids[0, g, 0] = target[g]
        ids[0, g, 1] = (target[g] + 3) % T.seg.m
        count[0, g] = 2
    # the expanded span's reconstructed tokens carry (almost) none of the mass its coarse entry would have had
    for g in range(Hkv):
        f = T.factors[g][target[g]]
        tok = ((f.UK * f.sK) @ f.VtK) @ q[0, g * G + 3] / np.sqrt(128.0)
        coarse = T.mean_K[g, target[g]] @ q[0, g * G + 3] / np.sqrt(128.0) + np.log(float(T.seg.span_len[target[g]]))
        assert tok.max() < coarse - 8.0
    _, worst = compare_attn(eng, 0, qd, ids, count, tabs, TOL_BF16)
    print("needle attention", "generic" if impl else "fused", worst)
    # and with the needle span NOT expanded its coarse entry does dominate: the output is ~ v_bar_s
    count0 = torch.zeros_like(count)
    out, _ = compare_attn(eng, 0, qd, ids, count0, tabs, TOL_BF16)
    o = out.float().cpu().numpy()
    for g in range(Hkv):
        assert rel_l2(o[0, g * G + 3], T.mean_V[g, target[g]]) < 1e-2
    eng.close()


# ---------------------------------------------------------------------------------------------------
# (d) sweeps: config 3 at batch 1 ... 64, config 4 at r = 8 and 32
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("batch", [1, 8, 16, 64])
def test_config3_ragged_batch_sweep(batch):
    spec = get_spec(3, batch=batch)
    lay = make_layouts(spec)
    eng = _engine(spec, lay, gen_device="cuda", prefetch=4)
    fused, why = eng.sekv_get_path()
    assert fused, why
    sample = sorted({0, batch // 2, batch - 1})
    tabs = _tables(eng, spec, factor_seqs=sample)
    q = make_queries(spec, 0, "cuda")[0]
    ids, count, _ = compare_route(eng, 0, q, spec.top_k, tabs)
    _, worst = compare_attn(eng, 0, q, ids, count, tabs, TOL_BF16, heads=[0, 5, 17, 31], seqs=sample)
    print(f"cfg3 B={batch}", worst)
    # the whole step (route + plan + attention in one launch per layer) on the same query
    out = torch.zeros((1, batch, spec.n_q_heads, 128), dtype=eng.out_dtype, device="cuda")
    eng.sekv_decode_step(q[None].contiguous(), spec.top_k, out)
    torch.cuda.synchronize()
    qn = to_np(q)
    ids2, count2 = eng.sekv_last_zoom_ids(0)
    for b in sample:
        T = tabs[b]
        zoom = [[int(x) for x in ids2[b, g, :int(count2[b, g])].cpu().numpy()] for g in range(spec.n_kv_heads)]
        ref, _ = O.decode_attn(qn[b], T, zoom, heads=[0, 5, 17, 31])
        got = out[0, b].float().cpu().numpy()
        assert rel_l2(got[[0, 5, 17, 31]], ref[[0, 5, 17, 31]]) <= TOL_BF16["rel_l2"]
    eng.close()


@pytest.mark.parametrize("rank", [8, 32])
def test_config4_rank_sweep_8_and_32(rank):
    spec = get_spec(4, rank=rank, top_k=-1)
    lay = make_layouts(spec)
    li = make_layer_inputs(spec, lay, 0)
    eng = _engine(spec, lay, li)
    assert eng.sekv_get_path()[0]
    tabs = _tables(eng, spec)
    q = make_queries(spec, 0, "cuda")[0]
    heads = [0, 6, 7, 13, 20, 27]
    for k in (0, 8, 64, -1):
        ids, count, _ = compare_route(eng, 0, q, k, tabs)
        _, worst = compare_attn(eng, 0, q, ids, count, tabs, TOL_BF16, heads=heads)
        print(f"cfg4 r={rank} k={k}", worst)
    eng.close()


# ---------------------------------------------------------------------------------------------------
# (e) local window (Eq. 17): the last w tokens stay at full resolution
# ---------------------------------------------------------------------------------------------------
def test_window_512_dense_build():
    spec = get_spec(1).with_(contexts=(9000,), window=512)
    lay = make_layouts(spec)
    li = make_layer_inputs(spec, lay, 0, dense=True)
    eng = _engine(spec, lay, li, mode="dense")
    tabs = _tables(eng, spec)
    T = tabs[0]
    ref = oracle_tables(spec, lay, li, 0, mode="dense")
    assert np.array_equal(T.seg.span_start, ref.seg.span_start) and np.array_equal(T.seg.span_len, ref.seg.span_len)
    assert np.array_equal(T.seg.pool_pos, ref.seg.pool_pos)
    n = lay[0].n
    assert set(range(n - 512, n)) <= set(int(x) for x in T.seg.pool_pos)           # the window is full resolution
    assert (T.seg.span_start + T.seg.span_len <= n - 512).all()
    assert T.seg.A > lay[0].A                                                      # more pool tokens than the planted anchors
    assert np.array_equal(T.full_K, ref.full_K) and np.array_equal(T.full_V, ref.full_V)
    q = make_queries(spec, 0, "cuda")[0]
    ids, count, _ = compare_route(eng, 0, q, spec.top_k, tabs)
    compare_attn(eng, 0, q, ids, count, tabs, TOL_BF16)
    eng.close()


# ---------------------------------------------------------------------------------------------------
# (f) CUDA-graph replay: one captured graph, new queries copied in place
# ---------------------------------------------------------------------------------------------------
def test_graph_replay_in_place_queries_single_graph():
    from paper_2606_31145_b200.export import export_tables
    spec = get_spec(1).sharp().with_(n_layers=3, contexts=(14000,))
    lay = make_layouts(spec)
    eng = _engine(spec, lay, prefetch=4, use_graph=1, out_dtype="bf16")
    L, Hq, Hkv = spec.n_layers, spec.n_q_heads, spec.n_kv_heads
    tabs = [tables_from_export(export_tables(eng, l, 0), Hq, Hkv, spec.route_dim) for l in range(L)]
    q = make_queries(spec, 0, "cuda")
    q_cur = torch.empty_like(q)
    out = torch.zeros((L, 1, Hq, 128), dtype=eng.out_dtype, device="cuda")
    for step in range(5):
        q_cur.copy_(q)                                        # same tensor every step: the graph is replayed
        eng.sekv_decode_step(q_cur, spec.top_k, out)
        torch.cuda.synchronize()
        assert eng.sekv_graph_count() == 1
        qn = to_np(q)
        out_h = out.float().cpu().numpy().astype(np.float64)
        for l in range(L):
            ids, count = eng.sekv_last_zoom_ids(l)
            torch.cuda.synchronize()
            R = O.route(qn[l, 0], tabs[l].W, tabs[l].route_K, tabs[l].seg.span_len, Hkv, spec.top_k)
            zoom = []
            for g in range(Hkv):
                c = int(count[0, g])
                check_ids(ids[0, g, :c].cpu().numpy(), R.ids[g], R.group_logit[g])
                zoom.append([int(x) for x in ids[0, g, :c].cpu().numpy()])
            ref, _ = O.decode_attn(qn[l, 0], tabs[l], zoom, heads=[0, 9, 31])
            assert rel_l2(out_h[l, 0, [0, 9, 31]], ref[[0, 9, 31]]) <= TOL_BF16["rel_l2"], (step, l)
        q = next_queries_ar1(spec, q, step + 1, 0.8)
    st = eng.sekv_get_stats()
    assert st["layer_steps"] == 5 * L and st["cache_hits"] > 0 and st["prefetched_spans"] > 0
    eng.close()


# ---------------------------------------------------------------------------------------------------
# (g) nothing switches kernels silently
# ---------------------------------------------------------------------------------------------------
def test_path_is_reported():
    spec = get_spec(1).with_(contexts=(6000,))
    lay = make_layouts(spec)
    li = make_layer_inputs(spec, lay, 0)
    eng = _engine(spec, lay, li)
    assert eng.sekv_get_path() == (True, "")
    eng.close()
    eng = _engine(spec, lay, li, impl=1)
    fused, why = eng.sekv_get_path()
    assert not fused and "impl" in why
    eng.close()
    spec0 = get_spec(0)
    lay0 = make_layouts(spec0)
    eng = _engine(spec0, lay0, make_layer_inputs(spec0, lay0, 0))
    fused, why = eng.sekv_get_path()
    assert not fused and "fp32" in why
    eng.close()
