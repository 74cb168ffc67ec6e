"""GPU parity on the degenerate sequences the method has, mixed into one ragged batch with a normal sequence:
a sequence without any span (every run is shorter than L_min: all tokens stay at full resolution),
a sequence that is ONE span with no full-resolution token (constant surprisal: sigma = 0, no boundary, L55), and a
short sequence with fewer spans than the zoom cap k (Eq. 9 / cap L123: the zoom set is every span).  Route, attention
on caller-supplied zoom sets and the whole step are compared with the oracle on the library's exported tables."""
from __future__ import annotations

import numpy as np
import pytest
import torch

from oracle import sekv_oracle as O
from tests.gpu_common import TOL_BF16, compare_attn, compare_route, tables_from_export
from tests.helpers import rel_l2, to_np
from workloads import SequenceLayout, get_spec, make_layouts, make_queries

pytestmark = pytest.mark.gpu


def _layout(n, H, spans, pool):
    return SequenceLayout(n=n, H=np.asarray(H, dtype=np.float32),
                          planted_span_start=np.asarray([s for s, _ in spans], dtype=np.int64),
                          planted_span_len=np.asarray([l for _, l in spans], dtype=np.int64),
                          planted_pool_pos=np.asarray(pool, dtype=np.int64))


def _degenerate_layouts(spec):
    rng = np.random.Generator(np.random.PCG64(spec.seed ^ 0xED6E))
    normal = make_layouts(spec.with_(contexts=(8192,)))[0]
    # (1) no span: runs of 10 low-surprisal tokens (< L_min = 16) between single high tokens -> all 48 tokens pooled
    H1 = np.ones(48, dtype=np.float32)
    H1[10::11] = 9.0
    no_span = _layout(48, H1, [], list(range(48)))
    # (2) one span, no pool token: constant surprisal -> sigma = 0, H_t > mu never holds, one run of 600 tokens
    one_span = _layout(600, np.ones(600, dtype=np.float32), [(0, 600)], [])
    # (3) three spans (20, 30, 17 tokens) and five anchors: fewer spans than k = 16
    H3, spans3, pool3, pos = [], [], [], 0
    for ln, na in ((20, 2), (30, 2), (17, 1)):
        H3 += list(rng.uniform(0.5, 1.5, size=ln)); spans3.append((pos, ln)); pos += ln
        H3 += list(8.0 + rng.uniform(0.0, 1.0, size=na)); pool3 += list(range(pos, pos + na)); pos += na
    few = _layout(pos, H3, spans3, pool3)
    return [normal, no_span, one_span, few]


@pytest.mark.parametrize("impl", [0, 1])
def test_degenerate_sequences_in_one_batch(impl):
    from paper_2606_31145_b200 import engine as E
    from paper_2606_31145_b200.export import export_tables
    base = get_spec(3, batch=4).sharp()
    lay = _degenerate_layouts(base)
    spec = base.with_(contexts=tuple(l.n for l in lay))
    eng = E.create_engine(spec, lay, gen_device="cuda", prefetch=4, impl=impl)
    fused, why = eng.sekv_get_path()
    assert bool(fused) == (impl == 0), why
    tabs = [tables_from_export(export_tables(eng, 0, b, True), spec.n_q_heads, spec.n_kv_heads, spec.route_dim)
            for b in range(4)]
    # the library segments these sequences the way they were planted
    assert [T.seg.m for T in tabs] == [lay[0].m, 0, 1, 3]
    assert [len(T.seg.pool_pos) for T in tabs] == [lay[0].A, 48, 0, 5]
    q = make_queries(spec, 0, "cuda")[0]
    ids, count, refs = compare_route(eng, 0, q, spec.top_k, tabs)
    cnt = count.cpu().numpy()
    assert (cnt[1] == 0).all() and (cnt[2] == 1).all() and (cnt[3] == 3).all() and (cnt[0] == spec.top_k).all()
    _, worst = compare_attn(eng, 0, q, ids, count, tabs, TOL_BF16)
    _, worst0 = compare_attn(eng, 0, q, ids, torch.zeros_like(count), tabs, TOL_BF16)     # nothing zoomed
    print("degenerate batch", impl, worst, worst0)
    # the whole step on the same query, twice (the second step runs on a warm factor cache)
    out = torch.zeros((1, 4, spec.n_q_heads, 128), dtype=eng.out_dtype, device="cuda")
    qn = to_np(q)
    for _ in range(2):
        eng.sekv_decode_step(q[None].contiguous(), spec.top_k, out)
        torch.cuda.synchronize()
        ids2, count2 = eng.sekv_last_zoom_ids(0)
        for b, T in enumerate(tabs):
            zoom = [[int(x) for x in ids2[b, g, :int(count2[b, g])].cpu().numpy()] for g in range(spec.n_kv_heads)]
            ref, _ = O.decode_attn(qn[b], T, zoom)
            got = out[0, b].float().cpu().numpy()
            assert rel_l2(got, ref) <= TOL_BF16["rel_l2"], (b, rel_l2(got, ref))
            assert float(np.abs(got - ref).max()) <= TOL_BF16["max_abs"]
    eng.close()


def _max_span_spec(n_spans):
    # spans of exactly L_min = 16 tokens, two anchors after each (the last span takes the two leftover tokens too)
    return get_spec(1).sharp().with_(contexts=(18 * n_spans,), len_lo=16, len_hi=16, anchors_per_span=2)


def test_maximum_spans_per_sequence():
    """SEKV_MAX_SPANS_PER_SEQ = 8192 spans in ONE sequence (the most the span tables of a sequence hold): routing over
    8192 summaries per head and the top-k select over them, attention with 16 of them expanded."""
    from paper_2606_31145_b200 import engine as E
    from paper_2606_31145_b200.export import export_tables
    spec = _max_span_spec(8192)
    lay = make_layouts(spec)
    assert lay[0].m == 8192 and lay[0].A == 2 * 8191
    eng = E.create_engine(spec, lay, gen_device="cuda", prefetch=4)
    fused, why = eng.sekv_get_path()
    print("8192 spans: fused =", bool(fused), why)
    T = tables_from_export(export_tables(eng, 0, 0, True), spec.n_q_heads, spec.n_kv_heads, spec.route_dim)
    assert T.seg.m == 8192
    q = make_queries(spec, 0, "cuda")[0]
    ids, count, _ = compare_route(eng, 0, q, spec.top_k, [T])
    _, worst = compare_attn(eng, 0, q, ids, count, [T], TOL_BF16, heads=[0, 9, 22, 31])
    out = torch.zeros((1, 1, spec.n_q_heads, 128), dtype=eng.out_dtype, device="cuda")
    eng.sekv_decode_step(q[None].contiguous(), spec.top_k, out)
    torch.cuda.synchronize()
    ids2, count2 = eng.sekv_last_zoom_ids(0)
    zoom = [[int(x) for x in ids2[0, g, :int(count2[0, g])].cpu().numpy()] for g in range(spec.n_kv_heads)]
    ref, _ = O.decode_attn(to_np(q)[0], T, zoom, heads=[0, 9, 22, 31])
    got = out[0, 0].float().cpu().numpy()
    assert rel_l2(got[[0, 9, 22, 31]], ref[[0, 9, 22, 31]]) <= TOL_BF16["rel_l2"]
    print("8192 spans", worst)
    eng.close()


def test_one_span_more_than_the_maximum_is_refused():
    from paper_2606_31145_b200 import binding as B
    from paper_2606_31145_b200 import engine as E
    spec = _max_span_spec(8193)
    lay = make_layouts(spec)
    assert lay[0].m == 8193
    with pytest.raises(B.SekvError) as ei:
        E.create_engine(spec, lay, gen_device="cuda", prefetch=4)
    assert ei.value.status in (B.SEKV_UNSUPPORTED, B.SEKV_INVALID_ARG) and "8192" in str(ei.value)


def test_maximum_span_length_and_rank():
    """Spans of SEKV_MAX_SPAN_LEN = 1024 tokens with rank SEKV_MAX_RANK = 64 factors (the largest blob the store
    holds: 289 KB, read in many windows), 28 / 4 heads (G = 7), the first step with every expansion a demand miss."""
    from paper_2606_31145_b200 import engine as E
    from paper_2606_31145_b200.export import export_tables
    spec = get_spec(4, rank=64, top_k=8).sharp().with_(contexts=(20 * 1028 - 4,), len_lo=1024, len_hi=1024)
    lay = make_layouts(spec)
    assert lay[0].m == 20 and int(lay[0].planted_span_len.min()) == 1024 and int(lay[0].planted_span_len.max()) == 1024
    eng = E.create_engine(spec, lay, gen_device="cuda", prefetch=2)
    fused, why = eng.sekv_get_path()
    assert fused, why
    T = tables_from_export(export_tables(eng, 0, 0, True), spec.n_q_heads, spec.n_kv_heads, spec.route_dim)
    q = make_queries(spec, 0, "cuda")[0]
    ids, count, _ = compare_route(eng, 0, q, spec.top_k, [T])
    out = torch.zeros((1, 1, spec.n_q_heads, 128), dtype=eng.out_dtype, device="cuda")
    for step in range(2):                       # step 0: all demand misses (host store over PCIe), step 1: all hits
        eng.sekv_decode_step(q[None].contiguous(), spec.top_k, out)
        torch.cuda.synchronize()
        ids2, count2 = eng.sekv_last_zoom_ids(0)
        zoom = [[int(x) for x in ids2[0, g, :int(count2[0, g])].cpu().numpy()] for g in range(spec.n_kv_heads)]
        ref, _ = O.decode_attn(to_np(q)[0], T, zoom)
        got = out[0, 0].float().cpu().numpy()
        assert rel_l2(got, ref) <= TOL_BF16["rel_l2"], (step, rel_l2(got, ref))
        assert float(np.abs(got - ref).max()) <= TOL_BF16["max_abs"]
    st = eng.sekv_get_stats()
    assert st["cache_misses"] >= 8 * spec.n_kv_heads and st["cache_hits"] >= 8 * spec.n_kv_heads
    eng.close()
