"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element, on the
seeded workloads of BASELINE.json configs 0, 1, 3, 4 (config 2 is in test_gpu_config2.py).

Protocol: the library builds its tables from the generator's tensors; the tables are
exported and (1) compared with the oracle's own construction, (2) fed to the oracle's routing and
attention, whose results the library must match on the same queries and zoom sets."""
from __future__ import annotations

import numpy as np
import pytest
import torch

from oracle import sekv_oracle as O
from tests.gpu_common import (TOL_BF16, TOL_F32, assert_stored_close, compare_attn, compare_route,
                              tables_from_export)
from tests.helpers import oracle_tables, rel_l2, to_np
from workloads import get_spec, make_layer_inputs, make_layouts, make_queries

pytestmark = pytest.mark.gpu


def _engine(spec, lay, li=None, **kw):
    from paper_2606_31145_b200 import engine as E
    return E.create_engine(spec, lay, layer_inputs=None if li is None else [li], **kw)


def _exported(eng, spec, layer=0, with_factors=True):
    from paper_2606_31145_b200.export import export_tables
    raw = [export_tables(eng, layer, b, with_factors) for b in range(eng.n_seqs)]
    return [tables_from_export(ex, spec.n_q_heads, spec.n_kv_heads, spec.route_dim) for ex in raw], raw


def _check_build_against_oracle(spec, lay, li, tabs, raw, mode="prefactored"):
    for b, (T, ex) in enumerate(zip(tabs, raw)):
        ref = oracle_tables(spec, lay, li, b, mode=mode)
        assert np.array_equal(T.seg.span_start, ref.seg.span_start)        # span offsets exact
        assert np.array_equal(T.seg.span_len, ref.seg.span_len)
        assert np.array_equal(T.seg.pool_pos, ref.seg.pool_pos)
        assert np.allclose(ex["ln_len"], np.log(ref.seg.span_len), atol=1e-6)
        assert np.array_equal(T.full_K, ref.full_K) and np.array_equal(T.full_V, ref.full_V)
        assert_stored_close(T.mean_K, ref.mean_K, spec.dtype, "k_bar")
        assert_stored_close(T.mean_V, ref.mean_V, spec.dtype, "v_bar")
        assert_stored_close(T.route_K, ref.route_K, spec.dtype, "K_bar", ulps=2.0)
        for g in range(spec.n_kv_heads):
            for s in range(0, T.seg.m, max(1, T.seg.m // 7)):
                f, fr = T.factors[g][s], ref.factors[g][s]
                assert ex["factors"][g][s]["pad_ok"]
                if mode == "prefactored":      # stored verbatim
                    for a in ("UK", "sK", "VtK", "UV", "sV", "VtV"):
                        assert np.array_equal(getattr(f, a), getattr(fr, a)), (a, g, s)
                else:                          # through the products only (sign / rotation freedom)
                    Kh = O.gated_reconstruction(f.UK, f.sK, f.VtK)
                    Kr = O.gated_reconstruction(fr.UK, fr.sK, fr.VtK)
                    assert rel_l2(Kh, Kr) < (2e-2 if spec.dtype == "bf16" else 2e-5), (g, s, rel_l2(Kh, Kr))
                    assert np.allclose(f.sK, fr.sK, rtol=2e-3 if spec.dtype == "bf16" else 2e-5, atol=1e-6 * fr.sK.max())


def test_config0_tiny_f32_build_route_attention():
    spec = get_spec(0)
    lay = make_layouts(spec)
    li = make_layer_inputs(spec, lay, 0)
    eng = _engine(spec, lay, li)
    tabs, raw = _exported(eng, spec)
    _check_build_against_oracle(spec, lay, li, tabs, raw)
    for step in range(2):
        q = make_queries(spec, step, "cuda")[0]
        ids, count, _ = compare_route(eng, 0, q, spec.top_k, tabs)
        compare_attn(eng, 0, q, ids, count, tabs, TOL_F32)
    eng.close()


@pytest.mark.parametrize("sharp", [False, True])
def test_config1_llama8b_32k(sharp):
    spec = get_spec(1)
    if sharp:
        spec = spec.sharp()
    lay = make_layouts(spec)
    li = make_layer_inputs(spec, lay, 0)
    eng = _engine(spec, lay, li)
    tabs, raw = _exported(eng, spec)
    _check_build_against_oracle(spec, lay, li, tabs, raw)
    q = make_queries(spec, 0, "cuda")[0]
    ids, count, _ = compare_route(eng, 0, q, spec.top_k, tabs)
    _, worst = compare_attn(eng, 0, q, ids, count, tabs, TOL_BF16)
    print("cfg1", "sharp" if sharp else "plain", worst)
    # a second step with a new query reuses cached factors where the zoom sets overlap
    q2 = make_queries(spec, 1, "cuda")[0]
    ids2, count2, _ = compare_route(eng, 0, q2, spec.top_k, tabs)
    compare_attn(eng, 0, q2, ids2, count2, tabs, TOL_BF16)
    st = eng.sekv_get_stats()
    assert st["cache_hits"] + st["cache_misses"] == st["zoomed_spans"] == 2 * 8 * 16
    assert st["cache_misses"] >= 8 * 16
    eng.close()


def test_config1_needle_top1_known_by_construction():
    """q aligned with one span's routing summary: its top-1 is known by construction."""
    spec = get_spec(1).sharp()
    lay = make_layouts(spec)
    li = make_layer_inputs(spec, lay, 0)
    eng = _engine(spec, lay, li)
    tabs, _ = _exported(eng, spec, with_factors=False)
    T = tabs[0]
    target = [(7 * g + 3) % T.seg.m for g in range(spec.n_kv_heads)]
    q = np.zeros((1, spec.n_q_heads, 128))
    G = spec.group
    for h in range(spec.n_q_heads):
        # q with W q = 40 * K_bar[h, target]: least-squares preimage through pinv(W)
        q[0, h] = np.linalg.pinv(T.W[h]) @ (40.0 * T.route_K[h, target[h // G]])
    qd = torch.from_numpy(q).to(torch.bfloat16).cuda()
    ids, count = eng.sekv_route(0, qd, 1)
    torch.cuda.synchronize()
    assert ids[0, :, 0].cpu().tolist() == target
    compare_route(eng, 0, qd, 4, tabs)
    eng.close()


@pytest.mark.parametrize("rank", [4, 16, 64])
def test_config4_stress_rank_by_topk(rank):
    """64K context, 28 q heads / 4 kv heads (G = 7): r x top-k in {0, 8, 64, all}; the all-zoomed case is
    checked against dense attention over K = U diag(S) V^T (torch SDPA, fp64) as well as the oracle."""
    spec = get_spec(4, rank=rank, top_k=-1)
    lay = make_layouts(spec)
    li = make_layer_inputs(spec, lay, 0)
    eng = _engine(spec, lay, li)
    tabs, raw = _exported(eng, spec)
    if rank == 16:
        _check_build_against_oracle(spec, lay, li, tabs, raw)
    q = make_queries(spec, 0, "cuda")[0]
    heads = [0, 6, 7, 13, 20, 27]
    for k in (0, 8, 64, -1):
        ids, count, _ = compare_route(eng, 0, q, k, tabs)
        out, worst = compare_attn(eng, 0, q, ids, count, tabs, TOL_BF16, heads=heads)
        print(f"cfg4 r={rank} k={k}", worst)
    # all spans zoomed + exact-rank factors == dense softmax attention over the original K/V
    T, l = tabs[0], lay[0]
    out_h = out.to(torch.float32).cpu().numpy().astype(np.float64)
    qn = to_np(q)
    for h in (0, 13, 27):
        g = h // spec.group
        K = np.zeros((l.n, 128)); V = np.zeros((l.n, 128))
        K[T.seg.pool_pos] = T.full_K[g]; V[T.seg.pool_pos] = T.full_V[g]
        for s in range(T.seg.m):
            a, ln = int(T.seg.span_start[s]), int(T.seg.span_len[s])
            f = T.factors[g][s]
            K[a:a + ln] = (f.UK * f.sK) @ f.VtK; V[a:a + ln] = (f.UV * f.sV) @ f.VtV
        ref = torch.nn.functional.scaled_dot_product_attention(
            torch.from_numpy(qn[0, h])[None, None, None], torch.from_numpy(K)[None, None],
            torch.from_numpy(V)[None, None])[0, 0, 0].numpy()
        assert rel_l2(out_h[0, h], ref) <= TOL_BF16["rel_l2"] and np.abs(out_h[0, h] - ref).max() <= TOL_BF16["max_abs"]
    eng.close()


def test_config3_ragged_batch():
    """Ragged batch (contexts 8K-64K in one launch): CSR span table and split-K load balance."""
    spec = get_spec(3, batch=4)
    lay = make_layouts(spec)
    li = make_layer_inputs(spec, lay, 0)
    eng = _engine(spec, lay, li)
    tabs, raw = _exported(eng, spec)
    _check_build_against_oracle(spec, lay, li, tabs[:2], raw[:2])
    q = make_queries(spec, 0, "cuda")[0]
    ids, count, _ = compare_route(eng, 0, q, spec.top_k, tabs)
    compare_attn(eng, 0, q, ids, count, tabs, TOL_BF16, heads=[0, 5, 17, 31])
    n_ctas, parts = eng.sekv_get_schedule()
    assert n_ctas >= 148 and parts >= 1
    eng.close()


def test_dense_build_svd_through_products():
    """sekv_build_spans (dense K/V -> truncated SVD on the GPU) against the oracle's LAPACK SVD."""
    for cid, ctx in ((0, 2500), (1, 6000)):
        spec = get_spec(cid).with_(contexts=(ctx,))
        lay = make_layouts(spec)
        li = make_layer_inputs(spec, lay, 0, dense=True)
        eng = _engine(spec, lay, li, mode="dense")
        tabs, raw = _exported(eng, spec)
        _check_build_against_oracle(spec, lay, li, tabs, raw, mode="dense")
        q = make_queries(spec, 0, "cuda")[0]
        ids, count, _ = compare_route(eng, 0, q, spec.top_k, tabs)
        compare_attn(eng, 0, q, ids, count, tabs, TOL_F32 if cid == 0 else TOL_BF16)
        eng.close()
