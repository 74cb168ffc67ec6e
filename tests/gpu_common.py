"""Shared pieces of the GPU parity tests: build an engine from a seeded workload, turn the
library's exported tables into oracle Tables, and the comparison rules of BASELINE.json."""
from __future__ import annotations

from typing import List, Optional, Sequence

import numpy as np
import torch

from oracle import sekv_oracle as O
from tests.helpers import check_ids, rel_l2, to_np

# BASELINE.json north_star tolerances
TOL_BF16 = dict(rel_l2=2e-3, max_abs=1e-2, lse=2e-3)
TOL_F32 = dict(rel_l2=1e-5, max_abs=1e-5, lse=1e-4)      # SURVEY.md 8(c) proposal for fp32 storage


def tables_from_export(ex: dict, n_q_heads: int, n_kv_heads: int, route_dim: int) -> O.Tables:
    seg = O.Segmentation(n=ex["n"], pool_pos=ex["pool_pos"], span_start=ex["span_start"], span_len=ex["span_len"])
    factors = []
    for row in ex.get("factors", []):
        factors.append([O.SpanFactors(UK=f["UK"], sK=f["sK"], VtK=f["VtK"], UV=f["UV"], sV=f["sV"], VtV=f["VtV"])
                        for f in row])
    return O.Tables(n_q_heads=n_q_heads, n_kv_heads=n_kv_heads, head_dim=128, route_dim=route_dim, seg=seg,
                    full_K=ex["full_K"], full_V=ex["full_V"], mean_K=ex["mean_K"], mean_V=ex["mean_V"],
                    route_K=ex["route_K"], W=ex["W"], factors=factors)


def ulp_bf16(x: np.ndarray) -> np.ndarray:
    """Spacing of bf16 numbers at |x| (8 significand bits)."""
    ax = np.maximum(np.abs(x), 2.0 ** -126)
    return 2.0 ** (np.floor(np.log2(ax)) - 7)


def assert_stored_close(got: np.ndarray, ref: np.ndarray, dtype: str, what: str, ulps: float = 1.0):
    """Stored summaries must agree with the oracle's to within one storage ulp:
    the library accumulates in fp32 and the oracle in fp64 before rounding."""
    if dtype == "bf16":
        tol = ulps * ulp_bf16(ref) + 1e-30
        # near zero, cancellation in the fp32 accumulation is relative to the row's magnitude
        tol = np.maximum(tol, 2e-6 * np.abs(ref).max())
    else:
        # fp32 storage: fp32 accumulation of up to |S| products vs the oracle's fp64
        tol = 1e-5 * np.abs(ref) + 5e-6 * np.abs(ref).max() + 1e-30
    bad = np.abs(got - ref) > tol
    assert not bad.any(), f"{what}: {bad.sum()} of {bad.size} differ, worst {np.abs(got - ref).max():.3e}"


def compare_route(eng, layer: int, q_dev: torch.Tensor, k: int, tables: Sequence[O.Tables], tau=None,
                  logit_tol: float = 2e-5):
    """sekv_route vs the oracle on identical stored tables: logits and alpha element-wise, ids by
    the tie rule of BASELINE.json."""
    cfg = eng.cfg
    m_tot = sum(t.seg.m for t in tables)
    logits = torch.zeros((cfg.n_q_heads, m_tot), dtype=torch.float32, device=eng.device)
    alpha = torch.zeros_like(logits)
    tau_dev = None if tau is None else torch.tensor(tau, dtype=torch.float32, device=eng.device)
    ids, count = eng.sekv_route(layer, q_dev, k, tau=tau_dev, logits=logits, alpha_tilde=alpha)
    torch.cuda.synchronize()
    ids_h, count_h = ids.cpu().numpy(), count.cpu().numpy()
    q = to_np(q_dev)
    s0 = 0
    refs = []
    for b, T in enumerate(tables):
        R = O.route(q[b], T.W, T.route_K, T.seg.span_len, cfg.n_kv_heads, k, tau=tau)
        refs.append(R)
        if T.seg.m:
            got = logits[:, s0:s0 + T.seg.m].cpu().numpy().astype(np.float64)
            assert np.abs(got - R.logit).max() < logit_tol * max(1.0, np.abs(R.logit).max()), \
                f"seq {b}: logits differ by {np.abs(got - R.logit).max():.3e}"
            ga = alpha[:, s0:s0 + T.seg.m].cpu().numpy().astype(np.float64)
            assert np.abs(ga - R.alpha).max() < 1e-5
        for g in range(cfg.n_kv_heads):
            c = int(count_h[b, g])
            assert c == len(R.ids[g]), (b, g, c, len(R.ids[g]))
            check_ids(ids_h[b, g, :c], R.ids[g], R.group_logit[g])
            assert (ids_h[b, g, c:] == -1).all()
        s0 += T.seg.m
    return ids, count, refs


def compare_attn(eng, layer: int, q_dev: torch.Tensor, ids: Optional[torch.Tensor], count: Optional[torch.Tensor],
                 tables: Sequence[O.Tables], tol: dict, heads: Optional[Sequence[int]] = None, seqs=None):
    """sekv_decode_attn vs the oracle's mixed-resolution attention on the SAME zoom sets."""
    cfg = eng.cfg
    lse = torch.zeros((eng.n_seqs, cfg.n_q_heads), dtype=torch.float32, device=eng.device)
    out = eng.sekv_decode_attn(layer, q_dev, ids, count, lse=lse)
    torch.cuda.synchronize()
    out_h = out.to(torch.float32).cpu().numpy().astype(np.float64)
    lse_h = lse.cpu().numpy().astype(np.float64)
    q = to_np(q_dev)
    ids_h = None if ids is None else ids.cpu().numpy()
    count_h = None if count is None else count.cpu().numpy()
    worst = dict(rel_l2=0.0, max_abs=0.0, lse=0.0)
    for b, T in enumerate(tables):
        if seqs is not None and b not in seqs:
            continue
        zoom = [[] for _ in range(cfg.n_kv_heads)]
        if ids_h is not None:
            for g in range(cfg.n_kv_heads):
                seen = []
                for s in ids_h[b, g, :int(count_h[b, g])]:
                    if 0 <= s < T.seg.m and int(s) not in seen:
                        seen.append(int(s))
                zoom[g] = seen
        ref, ref_lse = O.decode_attn(q[b], T, zoom, heads=heads)
        hs = list(range(cfg.n_q_heads)) if heads is None else list(heads)
        r = rel_l2(out_h[b, hs], ref[hs])
        a = float(np.abs(out_h[b, hs] - ref[hs]).max())
        worst["rel_l2"] = max(worst["rel_l2"], r)
        worst["max_abs"] = max(worst["max_abs"], a)
        fin = np.isfinite(ref_lse[hs])
        if fin.any():
            worst["lse"] = max(worst["lse"], float(np.abs(lse_h[b, hs][fin] - ref_lse[hs][fin]).max()))
        assert (np.isinf(lse_h[b, hs][~fin]) & (lse_h[b, hs][~fin] < 0)).all()
        assert r <= tol["rel_l2"], f"seq {b}: rel-L2 {r:.3e} > {tol['rel_l2']}"
        assert a <= tol["max_abs"], f"seq {b}: max-abs {a:.3e} > {tol['max_abs']}"
    assert worst["lse"] <= tol["lse"], worst
    return out, worst
