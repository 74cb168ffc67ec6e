"""sekv_export_tables: decode the library's stored tables (device arena + pinned host arena) into
plain numpy arrays in the paper's orientation, for tests and the timed CPU baseline.  Pure format
decoding driven by sekv_get_layout -- no arithmetic of the method."""
from __future__ import annotations

from typing import Dict, List

import numpy as np
import torch

from . import binding as B


def _view(arena: torch.Tensor, off: int, nbytes: int, dtype: torch.dtype) -> torch.Tensor:
    return arena[off:off + nbytes].view(dtype)


def _f64(t: torch.Tensor) -> np.ndarray:
    return t.detach().to(torch.float32).cpu().numpy().astype(np.float64)


def blob_sections(esize: int, ln: int, rk: int, rv: int) -> dict:
    """Byte offsets of a factor blob; mirrors the layout stated in sekv_internal.cuh:
    header [sK f32 rkp][sV f32 rvp][VtK rkp x 128][VV 128 x rvp], then lenp/16 chunks of 16 tokens,
    each [UK 16 x rkp][UVt rvp x 16]."""
    lenp = -(-ln // 16) * 16
    rkp = -(-max(rk, 1) // 8) * 8
    rvp = -(-max(rv, 1) // 8) * 8
    o = 0
    sec = {"lenp": lenp, "rkp": rkp, "rvp": rvp}
    sec["sk"] = o; o += rkp * 4
    sec["sv"] = o; o += rvp * 4
    sec["vtk"] = o; o += rkp * 128 * esize
    sec["vv"] = o; o += 128 * rvp * esize
    sec["chunks"] = o; o += lenp * (rkp + rvp) * esize
    sec["bytes"] = -(-o // 128) * 128
    return sec


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
        n_dir = lay.dir_layer_stride_elems
        dir_off = _view(dev, lay.dir_off + layer * n_dir * 8, n_dir * 8, torch.int64).view(Hkv, lay.spans_cap).cpu().numpy()
        dir_rank = _view(dev, lay.dir_rank + layer * n_dir * 4, n_dir * 4, torch.int32).view(Hkv, lay.spans_cap).cpu().numpy()
        host = eng.host_arena
        factors: List[List[dict]] = []
        for g in range(Hkv):
            row = []
            for s in range(s0, s1):
                ln = int(span_len[s]); rk = int(dir_rank[g, s]) & 0xff; rv = (int(dir_rank[g, s]) >> 8) & 0xff
                sec = blob_sections(es, ln, rk, rv)
                blob = host[int(dir_off[g, s]):int(dir_off[g, s]) + sec["bytes"]]
                sK = blob[sec["sk"]:sec["sk"] + sec["rkp"] * 4].view(torch.float32)
                sV = blob[sec["sv"]:sec["sv"] + sec["rvp"] * 4].view(torch.float32)
                VtK = blob[sec["vtk"]:sec["vtk"] + sec["rkp"] * 128 * es].view(st).view(sec["rkp"], 128)
                VV = blob[sec["vv"]:sec["vv"] + 128 * sec["rvp"] * es].view(st).view(128, sec["rvp"])
                ch = blob[sec["chunks"]:sec["chunks"] + sec["lenp"] * (sec["rkp"] + sec["rvp"]) * es].view(st)
                ch = ch.view(sec["lenp"] // 16, 16 * (sec["rkp"] + sec["rvp"]))
                UK = ch[:, :16 * sec["rkp"]].reshape(sec["lenp"], sec["rkp"])                       # [lenp][rkp]
                UVt = ch[:, 16 * sec["rkp"]:].reshape(sec["lenp"] // 16, sec["rvp"], 16).permute(1, 0, 2).reshape(sec["rvp"], sec["lenp"])
                row.append(dict(UK=_f64(UK[:ln, :rk]), sK=_f64(sK[:rk]), VtK=_f64(VtK[:rk]),
                                UV=_f64(UVt[:rv, :ln]).T.copy(), sV=_f64(sV[:rv]), VtV=_f64(VV[:, :rv]).T.copy(),
                                pad_ok=bool((UK[ln:].float() == 0).all() and (UVt[:, ln:].float() == 0).all()
                                            and (sK[rk:] == 0).all() and (sV[rv:] == 0).all())))
            factors.append(row)
        out["factors"] = factors
    return out
