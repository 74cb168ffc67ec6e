"""sekv_export_tables: the library's stored tables as plain numpy arrays in the paper's orientation, for
tests.  The row-major device tables are sliced out of the arena with the offsets of sekv_get_layout; the factor
blobs (stored in mma fragment order) are decoded by the library (sekv_export_span_factors).  No arithmetic of
the method."""
from __future__ import annotations

from typing import Dict, List

import numpy as np
import torch

from . import binding as B


def _view(arena: torch.Tensor, off: int, nbytes: int, dtype: torch.dtype) -> torch.Tensor:
    return arena[off:off + nbytes].view(dtype)


def _f64(t: torch.Tensor) -> np.ndarray:
    return t.detach().to(torch.float32).cpu().numpy().astype(np.float64)


def export_tables(eng: B.Sekv, layer: int, b: int, with_factors: bool = True) -> Dict:
    """Stored tables of sequence `b` at `layer` as float64 / int64 numpy arrays."""
    torch.cuda.synchronize(eng.device)
    lay = eng.sekv_get_layout()
    cfg = eng.cfg
    dev = eng.dev_arena
    st = eng.st_dtype
    es = eng.esize
    Bn, Hq, Hkv, dp = eng.n_seqs, cfg.n_q_heads, cfg.n_kv_heads, cfg.route_dim
    tok_off = _view(dev, lay.seq_tok_off, (Bn + 1) * 8, torch.int64).cpu().numpy()
    row_off = _view(dev, lay.seq_row_off, (Bn + 1) * 4, torch.int32).cpu().numpy()
    span_off = _view(dev, lay.seq_span_off, (Bn + 1) * 4, torch.int32).cpu().numpy()
    pool_cnt = _view(dev, lay.seq_pool_cnt, Bn * 4, torch.int32).cpu().numpy()
    m_tot, a_tot = int(span_off[Bn]), int(pool_cnt.sum())
    span_len = _view(dev, lay.span_len, m_tot * 4, torch.int32).cpu().numpy()
    span_tok = _view(dev, lay.span_tok_start, m_tot * 8, torch.int64).cpu().numpy()
    ln_len = _view(dev, lay.ln_len, m_tot * 4, torch.float32).cpu().numpy()
    pool_tok = _view(dev, lay.pool_tok, max(a_tot, 1) * 8, torch.int64).cpu().numpy()[:a_tot]
    s0, s1 = int(span_off[b]), int(span_off[b + 1])
    A = int(pool_cnt[b])
    p0 = int(pool_cnt[:b].sum())
    m = s1 - s0
    r0 = int(row_off[b])
    out = dict(n=int(tok_off[b + 1] - tok_off[b]), A=A, m=m,
               pool_pos=(pool_tok[p0:p0 + A] - tok_off[b]).astype(np.int64),
               span_start=(span_tok[s0:s1] - tok_off[b]).astype(np.int64),
               span_len=span_len[s0:s1].astype(np.int64), ln_len=ln_len[s0:s1].astype(np.float64))
    ent_k = _view(dev, lay.ent_k + layer * lay.ent_layer_stride, Hkv * lay.ent_head_stride, st).view(Hkv, lay.rows_cap, 128)
    ent_v = _view(dev, lay.ent_v + layer * lay.ent_layer_stride, Hkv * lay.ent_head_stride, st).view(Hkv, lay.rows_cap, 128)
    out["full_K"] = _f64(ent_k[:, r0:r0 + A]); out["full_V"] = _f64(ent_v[:, r0:r0 + A])
    out["mean_K"] = _f64(ent_k[:, r0 + A:r0 + A + m]); out["mean_V"] = _f64(ent_v[:, r0 + A:r0 + A + m])
    route = _view(dev, lay.route + layer * lay.route_layer_stride, Hq * lay.route_head_stride, st).view(Hq, lay.spans_cap, dp)
    out["route_K"] = _f64(route[:, s0:s1])
    out["W"] = _f64(_view(dev, lay.w + layer * lay.w_layer_stride, Hq * dp * 128 * es, st).view(Hq, dp, 128))
    if with_factors:
        # the blob layout (mma fragment order) is decoded by the library itself: sekv_export_span_factors
        factors: List[List[dict]] = []
        for g in range(Hkv):
            row = []
            for s in range(m):
                f = eng.sekv_export_span_factors(layer, b, g, s)
                row.append(dict(UK=f["UK"].astype(np.float64), sK=f["sK"].astype(np.float64),
                                VtK=f["VtK"].astype(np.float64), UV=f["UV"].astype(np.float64),
                                sV=f["sV"].astype(np.float64), VtV=f["VtV"].astype(np.float64), pad_ok=f["pad_ok"]))
            factors.append(row)
        out["factors"] = factors
    return out
