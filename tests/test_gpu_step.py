"""GPU parity of the whole-step entry point (sekv_decode_step): routing, residency plan, demand fetch,
side-stream prefetch, mixed-resolution attention and combine in ONE call per step, over several steps of an
AR(1) query stream so that the device factor cache goes through misses, hits, evictions and prefetches.
Every step's zoom sets and outputs are compared with the oracle on the exported tables."""
from __future__ import annotations

import numpy as np
import pytest
import torch

from oracle import sekv_oracle as O
from tests.gpu_common import TOL_BF16, tables_from_export
from tests.helpers import check_ids, rel_l2, to_np
from workloads import get_spec, make_layer_inputs, make_layouts, make_queries, next_queries_ar1

pytestmark = pytest.mark.gpu


def _run_steps(spec, n_steps, rho, heads=None, **cfg_kw):
    from paper_2606_31145_b200 import engine as E
    from paper_2606_31145_b200.export import export_tables
    lay = make_layouts(spec)
    eng = E.create_engine(spec, lay, **cfg_kw)
    tabs = [[tables_from_export(export_tables(eng, l, b), spec.n_q_heads, spec.n_kv_heads, spec.route_dim)
             for b in range(eng.n_seqs)] for l in range(spec.n_layers)]
    L, B, Hq, Hkv = spec.n_layers, spec.batch, spec.n_q_heads, spec.n_kv_heads
    q = make_queries(spec, 0, "cuda")
    out = torch.zeros((L, B, Hq, 128), dtype=eng.out_dtype, device="cuda")
    lse = torch.zeros((L, B, Hq), dtype=torch.float32, device="cuda")
    hs = list(range(Hq)) if heads is None else list(heads)
    worst = dict(rel_l2=0.0, max_abs=0.0, lse=0.0)
    for step in range(n_steps):
        eng.sekv_decode_step(q, spec.top_k, out, lse=lse)
        torch.cuda.synchronize()
        out_h = out.float().cpu().numpy().astype(np.float64)
        lse_h = lse.cpu().numpy().astype(np.float64)
        qn = to_np(q)
        for l in range(L):
            ids, count = eng.sekv_last_zoom_ids(l)
            torch.cuda.synchronize()
            ids_h, count_h = ids.cpu().numpy(), count.cpu().numpy()
            for b in range(B):
                T = tabs[l][b]
                R = O.route(qn[l, b], T.W, T.route_K, T.seg.span_len, Hkv, spec.top_k)
                zoom = []
                for g in range(Hkv):
                    c = int(count_h[b, g])
                    assert c == len(R.ids[g])
                    check_ids(ids_h[b, g, :c], R.ids[g], R.group_logit[g])
                    zoom.append([int(x) for x in ids_h[b, g, :c]])
                ref, ref_lse = O.decode_attn(qn[l, b], T, zoom, heads=hs)
                r = rel_l2(out_h[l, b, hs], ref[hs])
                a = float(np.abs(out_h[l, b, hs] - ref[hs]).max())
                e = float(np.abs(lse_h[l, b, hs] - ref_lse[hs]).max())
                worst = dict(rel_l2=max(worst["rel_l2"], r), max_abs=max(worst["max_abs"], a), lse=max(worst["lse"], e))
                assert r <= TOL_BF16["rel_l2"] and a <= TOL_BF16["max_abs"] and e <= TOL_BF16["lse"], (step, l, b, r, a, e)
        q = next_queries_ar1(spec, q, step + 1, rho)
    st = eng.sekv_get_stats()
    return eng, st, worst


@pytest.mark.parametrize("prefetch", [0, 8])
def test_step_config1_sharp_two_layers(prefetch):
    spec = get_spec(1).sharp().with_(n_layers=2, contexts=(20000,))
    eng, st, worst = _run_steps(spec, 5, 0.7, prefetch=prefetch)
    print("step cfg1", prefetch, worst, st)
    assert st["zoomed_spans"] == 5 * 2 * 8 * 16 == st["cache_hits"] + st["cache_misses"]
    assert st["layer_steps"] == 10
    assert st["cache_misses"] >= 2 * 8 * 16            # cold start
    assert st["cache_hits"] > 0                         # later steps reuse cached factors
    if prefetch:
        assert st["prefetched_spans"] > 0
    else:
        assert st["prefetched_spans"] == 0
    eng.close()


def test_step_prefetch_reduces_demand_misses():
    """Same stream with and without the speculative prefetch: identical outputs (checked against the oracle in
    both runs), fewer demand misses with it."""
    spec = get_spec(1).sharp().with_(contexts=(24000,))
    eng0, st0, _ = _run_steps(spec, 6, 0.9, heads=[0, 9, 31], prefetch=0, cache_ways=64)
    eng0.close()
    eng1, st1, _ = _run_steps(spec, 6, 0.9, heads=[0, 9, 31], prefetch=16, cache_ways=64)
    eng1.close()
    assert st1["cache_misses"] < st0["cache_misses"], (st0, st1)


@pytest.mark.parametrize("use_graph", [0, 1])
def test_step_four_layers_prefetch_two_launches_back(use_graph):
    """Three layers or more: a layer's prefetch candidates are copied by the kernel two launches later, before its
    dependency wait (layers 0 and 1 carry the last two layers' candidates of the previous step).  Every step of every
    layer against the oracle; the copies must have landed (prefetched spans turn into hits: fewer demand misses than
    without them), also after a caller reads the last two layers' caches between two steps (sekv_decode_attn on a
    layer whose copies are still pending runs them first)."""
    spec = get_spec(1).sharp().with_(n_layers=4, contexts=(18000,))
    eng0, st0, _ = _run_steps(spec, 6, 0.9, heads=[0, 9, 31], prefetch=0, cache_ways=64, use_graph=use_graph)
    eng0.close()
    eng1, st1, worst = _run_steps(spec, 6, 0.9, heads=[0, 9, 31], prefetch=8, cache_ways=64, use_graph=use_graph)
    print("step 4 layers", use_graph, worst, st0["cache_misses"], st1["cache_misses"], st1["prefetched_spans"])
    assert st1["layer_steps"] == 24 and st1["prefetched_spans"] > 0
    assert st1["cache_misses"] < st0["cache_misses"], (st0, st1)
    # between two steps: attention on the last two layers with the zoom sets of the last step (all hits now)
    from paper_2606_31145_b200.export import export_tables
    from tests.gpu_common import compare_attn
    q = make_queries(spec, 99, "cuda")
    for l in (2, 3):
        ids, count = eng1.sekv_last_zoom_ids(l)
        T = tables_from_export(export_tables(eng1, l, 0), spec.n_q_heads, spec.n_kv_heads, spec.route_dim)
        compare_attn(eng1, l, q[l], ids, count, [T], TOL_BF16, heads=[0, 9, 31])
    out = torch.zeros((4, 1, spec.n_q_heads, 128), dtype=eng1.out_dtype, device="cuda")
    eng1.sekv_decode_step(q, spec.top_k, out)
    torch.cuda.synchronize()
    qn = to_np(q)
    for l in range(4):
        ids, count = eng1.sekv_last_zoom_ids(l)
        T = tables_from_export(export_tables(eng1, l, 0), spec.n_q_heads, spec.n_kv_heads, spec.route_dim)
        zoom = [[int(x) for x in ids[0, g, :int(count[0, g])].cpu().numpy()] for g in range(spec.n_kv_heads)]
        ref, _ = O.decode_attn(qn[l, 0], T, zoom, heads=[0, 9, 31])
        assert rel_l2(out[l, 0].float().cpu().numpy()[[0, 9, 31]], ref[[0, 9, 31]]) <= TOL_BF16["rel_l2"], l
    eng1.close()


def test_step_ragged_batch_graph_replay():
    """Ragged batch (config 3, B = 3) through the CUDA-graph path: replays must see the new queries."""
    spec = get_spec(3, batch=3)
    eng, st, worst = _run_steps(spec, 3, 0.9, heads=[0, 13, 31], prefetch=4, use_graph=1)
    print("step cfg3", worst)
    assert st["layer_steps"] == 3
    eng.close()


def test_step_small_cache_evicts_lru():
    """cache_ways == k_cap + prefetch: every miss evicts; results stay exact."""
    spec = get_spec(1).sharp().with_(contexts=(16000,))
    eng, st, _ = _run_steps(spec, 4, 0.3, heads=[1, 18], prefetch=2, cache_ways=18)
    assert st["cache_misses"] > 8 * 16
    eng.close()


def test_step_config2_full_size_bench_configuration():
    """configs[2] at its full per-layer size (batch 4 x 128K context, r = 16, top-k = 32) in the launch
    configuration bench.py times (CUDA graph with programmatic dependent launches, speculative prefetch 8,
    bf16 output, AR(1) stream with rho = 0.99), two layers built: every step's zoom sets of every (sequence,
    kv head) and the outputs of a sample of query heads against the oracle."""
    spec = get_spec(2).with_(n_layers=2)
    eng, st, worst = _run_steps(spec, 3, 0.99, heads=[0, 5, 18, 31], prefetch=8, use_graph=1, out_dtype="bf16")
    print("step cfg2", worst, st)
    assert st["layer_steps"] == 6
    assert st["zoomed_spans"] == 3 * 2 * 4 * 8 * 32
    assert st["cache_hits"] > st["cache_misses"] // 2          # steps 2 and 3 reuse most of step 1's factors
    eng.close()


def test_item_trace_records_every_work_item():
    """sekv_set_trace: one 64-byte record per work item of a layer launch (plus one per group for the team's
    selection / plan), begin <= wait mark <= end, known kinds; switching it off leaves the outputs unchanged."""
    from paper_2606_31145_b200 import engine as E
    spec = get_spec(1).sharp().with_(contexts=(12000,))
    lay = make_layouts(spec)
    eng = E.create_engine(spec, lay)
    q = make_queries(spec, 0, "cuda")
    out0 = torch.zeros((1, 1, spec.n_q_heads, 128), dtype=torch.float32, device="cuda")
    out1 = torch.zeros_like(out0)
    eng.sekv_decode_step(q, spec.top_k, out0)
    buf = torch.zeros(16384 * 8, dtype=torch.int64, device="cuda")
    n = eng.sekv_set_trace(buf)
    assert n > 0
    eng.sekv_decode_step(q, spec.top_k, out1)
    torch.cuda.synchronize()
    groups = spec.batch * spec.n_kv_heads
    r = buf.cpu().numpy().reshape(-1, 8)
    rec = r[:n + groups]
    kind = rec[:, 0] & 0xFFFFFFFF
    assert (rec[:, 3] >= rec[:, 2]).all() and (rec[:, 2] > 0).all(), "every item has begin <= end stamps"
    assert (rec[:, 4] >= rec[:, 2]).all() and (rec[:, 4] <= rec[:, 3]).all(), "wait mark inside the item"
    assert set(int(k) for k in kind) <= set(range(7))
    assert int((kind == 2).sum()) == groups                     # one selection / plan per (sequence, kv head)
    assert (r[n + groups:] == 0).all()
    assert eng.sekv_set_trace(None) == n
    assert torch.equal(out0, out1)
    eng.close()


def test_soak_200_steps_graph_replay_misses_evictions_prefetch():
    """200 graph-replayed steps of configs[2] at its full per-layer size (two layers built) at rho = 0.9: ~12% demand
    misses per step, evictions, write-backs and prefetch copies carried by the next layer's kernel.  Every step: the
    cache statistics add up and the outputs are finite; the LAST step, reached through all that cache traffic, is
    compared with the oracle (every zoom set, sampled heads).  (compute-sanitizer is closed on the GPU pool: this
    is the long-run check of the kernel's polls, stamps and cross-proxy hand-offs.)"""
    from paper_2606_31145_b200 import engine as E
    from paper_2606_31145_b200.export import export_tables
    spec = get_spec(2).with_(n_layers=2)
    lay = make_layouts(spec)
    eng = E.create_engine(spec, lay, gen_device="cuda", prefetch=8, use_graph=1, out_dtype="bf16")
    assert eng.sekv_get_path()[0]
    L, B, Hq, Hkv = spec.n_layers, spec.batch, spec.n_q_heads, spec.n_kv_heads
    q = make_queries(spec, 0, "cuda")
    q_cur = torch.empty_like(q)
    out = torch.zeros((L, B, Hq, 128), dtype=eng.out_dtype, device="cuda")
    n_steps = 200
    for step in range(n_steps):
        q_cur.copy_(q)
        eng.sekv_decode_step(q_cur, spec.top_k, out)
        if step % 20 == 19 or step == n_steps - 1:
            torch.cuda.synchronize()
            assert torch.isfinite(out.float()).all(), step
            st = eng.sekv_get_stats()
            assert st["layer_steps"] == (step + 1) * L
            assert st["zoomed_spans"] == (step + 1) * L * B * Hkv * spec.top_k == st["cache_hits"] + st["cache_misses"]
        if step < n_steps - 1:
            q = next_queries_ar1(spec, q, step + 1, 0.9)
    assert eng.sekv_graph_count() == 1
    st = eng.sekv_get_stats()
    assert st["cache_misses"] > 200 * 50 and st["prefetched_spans"] > 0 and st["cache_hits"] > st["cache_misses"]
    qn = to_np(q)
    out_h = out.float().cpu().numpy().astype(np.float64)
    hs = [0, 5, 18, 31]
    for l in range(L):
        ids, count = eng.sekv_last_zoom_ids(l)
        torch.cuda.synchronize()
        ids_h, count_h = ids.cpu().numpy(), count.cpu().numpy()
        for b in (0, 3):
            T = tables_from_export(export_tables(eng, l, b), Hq, Hkv, spec.route_dim)
            R = O.route(qn[l, b], T.W, T.route_K, T.seg.span_len, Hkv, spec.top_k)
            zoom = []
            for g in range(Hkv):
                c = int(count_h[b, g])
                check_ids(ids_h[b, g, :c], R.ids[g], R.group_logit[g])
                zoom.append([int(x) for x in ids_h[b, g, :c]])
            ref, _ = O.decode_attn(qn[l, b], T, zoom, heads=hs)
            assert rel_l2(out_h[l, b, hs], ref[hs]) <= TOL_BF16["rel_l2"], (l, b)
            assert np.abs(out_h[l, b, hs] - ref[hs]).max() <= TOL_BF16["max_abs"]
    eng.close()
