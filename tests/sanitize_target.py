"""Target of the compute-sanitizer runs summarised under profiles/ (not a pytest module):

    compute-sanitizer --tool memcheck|racecheck|synccheck|initcheck python tests/sanitize_target.py [generic|fused]

generic: configs[0] (fp32, generic multi-kernel path): build, route, decode_attn.
fused:   a reduced configs[2] (2 layers, batch 2 x 16K context, bf16, fused layer kernel, no CUDA graph, prefetch 4):
         three decode steps of an AR(1) query stream (misses, hits, evictions, prefetch copies), then one explicit
         sekv_route + sekv_decode_attn on the last layer.
Outputs are checked for finiteness only: parity is the job of tests/test_gpu_*.py."""
from __future__ import annotations

import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch  # noqa: E402

from paper_2606_31145_b200 import engine as E  # noqa: E402
from workloads import get_spec, make_layouts, make_queries, next_queries_ar1  # noqa: E402


def run_generic():
    spec = get_spec(0)
    lay = make_layouts(spec)
    eng = E.create_engine(spec, lay)
    assert not eng.sekv_get_path()[0]
    q = make_queries(spec, 0, "cuda")[0]
    ids, count = eng.sekv_route(0, q, spec.top_k)
    out = eng.sekv_decode_attn(0, q, ids, count)
    torch.cuda.synchronize()
    assert torch.isfinite(out.float()).all()
    eng.close()


def run_fused():
    spec = get_spec(2).with_(n_layers=2, contexts=(16384, 16384))
    lay = make_layouts(spec)
    eng = E.create_engine(spec, lay, gen_device="cuda", prefetch=4, cache_ways=40, use_graph=0, out_dtype="bf16")
    fused, why = eng.sekv_get_path()
    assert fused, why
    q = make_queries(spec, 0, "cuda")
    out = torch.zeros((spec.n_layers, spec.batch, spec.n_q_heads, 128), dtype=eng.out_dtype, device="cuda")
    for step in range(3):
        eng.sekv_decode_step(q, spec.top_k, out)
        torch.cuda.synchronize()
        assert torch.isfinite(out.float()).all()
        q = next_queries_ar1(spec, q, step + 1, 0.7)
    ids, count = eng.sekv_route(1, q[1], spec.top_k)
    o = eng.sekv_decode_attn(1, q[1], ids, count)
    torch.cuda.synchronize()
    assert torch.isfinite(o.float()).all()
    st = eng.sekv_get_stats()
    assert st["cache_hits"] > 0 and st["cache_misses"] > 0
    eng.close()


if __name__ == "__main__":
    which = sys.argv[1] if len(sys.argv) > 1 else "fused"
    (run_generic if which == "generic" else run_fused)()
    print("sanitize target", which, "ok")
