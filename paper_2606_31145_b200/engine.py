"""Harness-side setup helper: size a sekv_config for a workload, create the handle, and stage the
generator's tensors through sekv_build_spans / sekv_build_spans_prefactored layer by layer.
No arithmetic of the method lives here -- only sizing, allocation and calls through the C ABI."""
from __future__ import annotations

from typing import Optional, Sequence

import numpy as np
import torch

from . import binding as B


def config_for(spec, layouts, *, k_cap: Optional[int] = None, cache_ways: Optional[int] = None,
               out_dtype: str = "f32", use_graph: int = 0, impl: int = 0, stage1_ctas: int = 0,
               r_max: Optional[int] = None, slack: float = 1.0, prefetch: int = 0, item_rows: int = 0,
               zoom_spans_per_item: int = 0, H_dev: Optional[torch.Tensor] = None, device="cuda:0"):
    """(sekv_config, pinned host bytes) for a batch.  Capacities come from sekv_build_sizes, i.e. from what a
    real caller has: the token counts and the surprisal tensor -- never from the generator's planted layout."""
    if H_dev is None:
        H_dev = surprisal_device(layouts, device)
    base = dict(n_layers=spec.n_layers, n_q_heads=spec.n_q_heads, n_kv_heads=spec.n_kv_heads, head_dim=spec.head_dim,
                route_dim=spec.route_dim, dtype=B.SEKV_BF16 if spec.dtype == "bf16" else B.SEKV_F32,
                out_dtype=B.SEKV_BF16 if out_dtype == "bf16" else B.SEKV_F32, alpha=spec.alpha, l_min=spec.l_min,
                r_max=r_max or spec.rank, window=spec.window, max_seqs=len(layouts))
    sz, _, _ = B.sekv_build_sizes(B.make_config(**base), seq_tok_off(layouts), H_dev)
    if k_cap is None:
        k_cap = sz.max_spans_per_seq if spec.top_k < 0 else spec.top_k
    if spec.top_k < 0:
        prefetch = 0
    if cache_ways is None:
        # SURVEY.md 8(c) reading 22: 4 x the per-step working set (and never fewer than two steps' zoom sets plus
        # prefetch candidates); at configs[2] that is 128 slots, inside the paper's 10% budget (L123)
        cache_ways = max(4 * k_cap, 2 * (k_cap + prefetch), 1) if spec.top_k >= 0 else max(k_cap, 1)
    cfg = B.make_config(
        **base, max_tokens_total=sz.tokens_total, max_spans_total=int(sz.spans_total * slack) + 1,
        max_full_total=int(sz.full_total * slack) + 1, max_span_len=min(1024, -(-max(sz.max_span_len, 16) // 16) * 16),
        k_cap=k_cap, cache_ways=max(cache_ways, 1), prefetch=prefetch, stage1_ctas=stage1_ctas, item_rows=item_rows,
        zoom_spans_per_item=zoom_spans_per_item, use_graph=use_graph, impl=impl)
    return cfg, int(sz.host_bytes)


def seq_tok_off(layouts) -> list:
    off = [0]
    for l in layouts:
        off.append(off[-1] + l.n)
    return off


def build_layer_prefactored(eng: B.Sekv, spec, layouts, li, H_dev: torch.Tensor):
    eng.sekv_build_spans_prefactored(
        li.layer, seq_tok_off(layouts), H_dev, rank_in=spec.rank, tokUK=li.tokUK, SK=li.SK, VtK=li.VtK,
        tokUV=li.tokUV, SV=li.SV, VtV=li.VtV, Kfull=li.Kfull, Vfull=li.Vfull, W=li.W, rank_k=li.rank_k,
        rank_v=li.rank_v, a_tot=sum(l.A for l in layouts), m_tot=sum(l.m for l in layouts))


def surprisal_device(layouts, device) -> torch.Tensor:
    return torch.from_numpy(np.concatenate([l.H for l in layouts]).astype(np.float32)).to(device)


def create_engine(spec, layouts, device="cuda:0", mode: str = "prefactored", gen_device: Optional[str] = None,
                  layer_inputs: Optional[Sequence] = None, **cfg_kw) -> B.Sekv:
    """Create a handle sized for `spec` and build every layer from the seeded generator."""
    from workloads import make_layer_inputs
    H_dev = surprisal_device(layouts, device)
    cfg, host_bytes = config_for(spec, layouts, H_dev=H_dev, device=device, **cfg_kw)
    eng = B.Sekv(cfg, host_bytes, device=device)
    gdev = gen_device or "cpu"
    for layer in range(spec.n_layers):
        li = layer_inputs[layer] if layer_inputs is not None else make_layer_inputs(
            spec, layouts, layer, device=gdev, dense=(mode == "dense"))
        li = to_device(li, eng.device)
        if mode == "dense":
            eng.sekv_build_spans(layer, seq_tok_off(layouts), H_dev, li.K, li.V, li.W, rank_cap=cfg.r_max)
        else:
            build_layer_prefactored(eng, spec, layouts, li, H_dev)
    return eng


def to_device(li, device):
    import dataclasses
    kw = {}
    for f in dataclasses.fields(li):
        v = getattr(li, f.name)
        kw[f.name] = v.to(device).contiguous() if isinstance(v, torch.Tensor) else v
    return type(li)(**kw)
