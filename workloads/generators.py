"""Seeded input synthesis for the SeKV hot path (recipe: DESIGN.md section 4).

Input synthesis ONLY.  Nothing here evaluates the paper's method: the segmentation rule, the
summaries, the routing score and the attention are implemented twice, independently, in
``oracle/`` (CPU, fp64) and in ``paper_2606_31145_b200/csrc`` (CUDA).  What this module does:

* draws span lengths and plants clusters of high-surprisal tokens after each span, so that the
  paper's boundary rule -- applied by whoever consumes ``H`` -- recovers the
  intended span table;
* draws, per (layer, kv head, span), random orthonormal factors ``U`` (|S| x r), ``V`` (d_h x r)
  and a decreasing spectrum ``S`` -- the generator's *definition* of the span's keys/values is
  ``K_S = U diag(S) V^T`` (BASELINE.json configs[0]);
* draws full-resolution (anchor) keys/values, routing projections ``W`` and queries.

Tensors are torch tensors on ``device`` in the storage dtype (bf16 or fp32): quantising the inputs
to the storage dtype is part of synthesising them -- a real model hands the cache bf16 tensors.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence

import numpy as np
import torch

from .configs import WorkloadSpec


def storage_torch_dtype(dtype: str) -> torch.dtype:
    return {"f32": torch.float32, "bf16": torch.bfloat16}[dtype]


# --------------------------------------------------------------------------------------------
# Layout: span lengths, anchor clusters, surprisal
# --------------------------------------------------------------------------------------------
@dataclass
class SequenceLayout:
    """One sequence's token layout as PLANTED by the generator (not as segmented by the method)."""
    n: int
    H: np.ndarray                      # [n] float32 surprisal
    planted_span_start: np.ndarray     # [m] int64, position of each planted span's first token
    planted_span_len: np.ndarray       # [m] int64
    planted_pool_pos: np.ndarray       # [A] int64, positions of full-resolution tokens (ascending)

    @property
    def m(self) -> int:
        return int(self.planted_span_len.shape[0])

    @property
    def A(self) -> int:
        return int(self.planted_pool_pos.shape[0])


def _one_layout(rng: np.random.Generator, n: int, spec: WorkloadSpec) -> SequenceLayout:
    H = np.empty(n, dtype=np.float32)
    starts: List[int] = []
    lens: List[int] = []
    pool: List[int] = []
    pos = 0
    na = spec.anchors_per_span
    while pos < n:
        ln = int(rng.integers(spec.len_lo, spec.len_hi + 1))
        if pos + ln + na >= n:
            ln = n - pos                           # last span truncated to fit, no trailing cluster
            H[pos:pos + ln] = rng.uniform(0.5, 1.5, size=ln).astype(np.float32)
            if ln >= spec.l_min:
                starts.append(pos)
                lens.append(ln)
            else:                                  # too short: full-resolution tokens (reading #5)
                pool.extend(range(pos, pos + ln))
            pos += ln
            break
        H[pos:pos + ln] = rng.uniform(0.5, 1.5, size=ln).astype(np.float32)
        starts.append(pos)
        lens.append(ln)
        pos += ln
        H[pos:pos + na] = (8.0 + rng.uniform(0.0, 1.0, size=na)).astype(np.float32)
        pool.extend(range(pos, pos + na))
        pos += na
    return SequenceLayout(n=n, H=H,
                          planted_span_start=np.asarray(starts, dtype=np.int64),
                          planted_span_len=np.asarray(lens, dtype=np.int64),
                          planted_pool_pos=np.asarray(pool, dtype=np.int64))


def make_layouts(spec: WorkloadSpec) -> List[SequenceLayout]:
    """Per-sequence layouts (layer-independent), seeded by ``spec.seed``."""
    out = []
    for b, n in enumerate(spec.contexts):
        rng = np.random.Generator(np.random.PCG64([spec.seed, 0x1A70, b]))
        out.append(_one_layout(rng, int(n), spec))
    return out


# --------------------------------------------------------------------------------------------
# Per-layer tensors
# --------------------------------------------------------------------------------------------
@dataclass
class LayerInputs:
    """Inputs of one layer for the whole batch.  Token axes are the concatenation of the batch's
    sequences; span axes the concatenation of their planted spans; pool axes likewise."""
    layer: int
    # prefactored form ------------------------------------------------------------------------
    tokUK: torch.Tensor      # [H_kv, sum_n, r]   storage dtype; row t = left-factor row of token t
    SK: torch.Tensor         # [H_kv, m_tot, r]   float32, descending, zero beyond rank
    VtK: torch.Tensor        # [H_kv, m_tot, r, d] storage dtype (right factor, transposed)
    tokUV: torch.Tensor
    SV: torch.Tensor
    VtV: torch.Tensor
    rank_k: torch.Tensor     # [H_kv, m_tot] int32 = min(r, |S|)
    rank_v: torch.Tensor
    Kfull: torch.Tensor      # [H_kv, A_tot, d]   storage dtype, pool tokens in position order
    Vfull: torch.Tensor
    W: torch.Tensor          # [H_q, d', d]       storage dtype
    # dense form (only when asked) --------------------------------------------------------------
    K: Optional[torch.Tensor] = None   # [H_kv, sum_n, d] storage dtype
    V: Optional[torch.Tensor] = None
    # generator-side float64 singular values kept for tests that want the exact spectrum
    extras: dict = field(default_factory=dict)


def _gen(device, *seed_words) -> torch.Generator:
    g = torch.Generator(device=device)
    s = 0
    for w in seed_words:                     # simple deterministic mix into 63 bits
        s = (s * 0x9E3779B97F4A7C15 + int(w) + 0x632BE59BD9B4E019) & 0x7FFFFFFFFFFFFFFF
    g.manual_seed(s)
    return g


def _orthonormal_columns(a: torch.Tensor) -> torch.Tensor:
    """Orthonormalise the columns of each matrix of a batch [..., rows, cols].
    CPU: LAPACK QR.  CUDA: two passes of Cholesky-QR (same Q up to column signs, all batched)."""
    if not a.is_cuda:
        q, _ = torch.linalg.qr(a, mode="reduced")
        return q
    q = a.to(torch.float64)
    eye = torch.eye(a.shape[-1], device=a.device, dtype=torch.float64)
    for _ in range(2):
        g = q.transpose(-1, -2) @ q
        # tiny relative shift keeps near-singular Gram matrices factorisable; the 2nd pass removes its effect
        g = g + eye * (1e-13 * g.diagonal(dim1=-2, dim2=-1).sum(-1)[..., None, None])
        l = torch.linalg.cholesky(g)
        q = torch.linalg.solve_triangular(l, q.transpose(-1, -2), upper=False).transpose(-1, -2)
    return q.to(a.dtype)


def _span_factors(gen: torch.Generator, lens: torch.Tensor, rows_pad: int, r: int, device,
                  work_dtype) -> tuple:
    """For a batch of spans with lengths ``lens`` [m]: U [m, rows_pad, r] with orthonormal columns
    supported on the first len rows and first min(r, len) columns, and the rank [m]."""
    m = lens.shape[0]
    rank = torch.clamp(lens, max=r)
    a = torch.randn((m, rows_pad, r), generator=gen, device=device, dtype=work_dtype)
    row_ok = torch.arange(rows_pad, device=device)[None, :, None] < lens[:, None, None]
    col_ok = torch.arange(r, device=device)[None, None, :] < rank[:, None, None]
    a = a * (row_ok & col_ok)
    if int(lens.min()) < r:
        # columns j >= rank get a unit vector in a padded row so the batch stays full column rank;
        # they are orthogonal to the real columns (zero there) and are dropped after the QR
        j = torch.arange(r, device=device)
        extra = torch.zeros((m, rows_pad, r), device=device, dtype=work_dtype)
        extra[:, j, j] = 1.0
        a = a + extra * (~col_ok)
    q = _orthonormal_columns(a)
    q = q * (row_ok & col_ok)
    return q, rank


def _spectrum(gen: torch.Generator, m: int, r: int, rank: torch.Tensor, device, work_dtype):
    """S = sort_desc(|N(0,1)| * 1/i), i = 1..r, zero beyond the rank (BASELINE.json configs[0])."""
    i = torch.arange(1, r + 1, device=device, dtype=work_dtype)
    s = torch.randn((m, r), generator=gen, device=device, dtype=work_dtype).abs() / i
    s = s * (torch.arange(r, device=device)[None, :] < rank[:, None])
    s, _ = torch.sort(s, dim=-1, descending=True)
    return s


def make_routing_weights(spec: WorkloadSpec, layer: int, device="cpu") -> torch.Tensor:
    """W ~ N(0, 1/d_h) entries, [H_q, d', d_h]; trained W are not available."""
    g = _gen(device, spec.seed, 0x3A77, layer)
    w = torch.randn((spec.n_q_heads, spec.route_dim, spec.head_dim), generator=g, device=device,
                    dtype=torch.float32)
    w = w * (spec.scale_w / float(spec.head_dim) ** 0.5)
    return w.to(storage_torch_dtype(spec.dtype))


def make_layer_inputs(spec: WorkloadSpec, layouts: Sequence[SequenceLayout], layer: int,
                      device="cpu", dense: bool = False, rows_pad: Optional[int] = None) -> LayerInputs:
    """All inputs of one layer.  ``dense=True`` also materialises K, V = U diag(S) V^T at the span
    tokens (BASELINE.json configs[0]: "per span K,V = U.diag(S).Vt") and the anchors elsewhere."""
    dev = torch.device(device)
    st = storage_torch_dtype(spec.dtype)
    work = torch.float32 if dev.type == "cuda" else torch.float64
    d, r, hk = spec.head_dim, spec.rank, spec.n_kv_heads
    lens_np = np.concatenate([l.planted_span_len for l in layouts]) if layouts else np.zeros(0, np.int64)
    m_tot = int(lens_np.shape[0])
    n_tot = int(sum(l.n for l in layouts))
    a_tot = int(sum(l.A for l in layouts))
    lens = torch.from_numpy(lens_np).to(dev)
    if rows_pad is None:
        rows_pad = int(max(int(lens_np.max()) if m_tot else 1, r))

    # token index of every (span, row-in-span) pair, for scattering padded U rows to token rows
    tok_base = 0
    span_tok_start = []
    for l in layouts:
        span_tok_start.append(l.planted_span_start + tok_base)
        tok_base += l.n
    span_tok_start = torch.from_numpy(np.concatenate(span_tok_start) if layouts else np.zeros(0, np.int64)).to(dev)
    j = torch.arange(rows_pad, device=dev)
    row_ok = j[None, :] < lens[:, None]                            # [m, rows_pad]
    tok_of = (span_tok_start[:, None] + j[None, :])[row_ok]        # [sum len]

    def one_side(tag: int, scale: float):
        tokU = torch.zeros((hk, n_tot, r), device=dev, dtype=st)
        S = torch.empty((hk, m_tot, r), device=dev, dtype=torch.float32)
        Vt = torch.empty((hk, m_tot, r, d), device=dev, dtype=st)
        rank = torch.empty((hk, m_tot), device=dev, dtype=torch.int32)
        dense_x = torch.zeros((hk, n_tot, d), device=dev, dtype=st) if dense else None
        for g in range(hk):
            gen = _gen(dev, spec.seed, 0xFAC7, layer, tag, g)
            U, rk = _span_factors(gen, lens, rows_pad, r, dev, work)              # [m, rows_pad, r]
            Vm, _ = _span_factors(gen, torch.full_like(lens, d), d, r, dev, work)  # [m, d, r]
            Vm = Vm * (torch.arange(r, device=dev)[None, None, :] < rk[:, None, None])
            s = _spectrum(gen, m_tot, r, rk, dev, work) * scale
            U_st = U.to(st)
            Vt_st = Vm.transpose(1, 2).contiguous().to(st)
            tokU[g, tok_of] = U_st[row_ok]
            S[g] = s.to(torch.float32)
            Vt[g] = Vt_st
            rank[g] = rk.to(torch.int32)
            if dense:
                x = (U * s[:, None, :]) @ Vm.transpose(1, 2)          # [m, rows_pad, d] from UNROUNDED factors
                dense_x[g, tok_of] = x[row_ok].to(st)
        return tokU, S, Vt, rank, dense_x

    tokUK, SK, VtK, rank_k, Kd = one_side(1, spec.scale_sk)
    tokUV, SV, VtV, rank_v, Vd = one_side(2, spec.scale_sv)

    # full-resolution (anchor / short-run) tokens: N(0, sigma), sigma = 1/sqrt(d_h)
    gen = _gen(dev, spec.seed, 0xA2C4, layer)
    sig = 1.0 / float(d) ** 0.5
    Kfull = (torch.randn((hk, a_tot, d), generator=gen, device=dev, dtype=torch.float32)
             * (sig * spec.scale_anchor_k)).to(st)
    Vfull = (torch.randn((hk, a_tot, d), generator=gen, device=dev, dtype=torch.float32) * sig).to(st)
    if dense:
        tok_base = 0
        pool_tok = []
        for l in layouts:
            pool_tok.append(l.planted_pool_pos + tok_base)
            tok_base += l.n
        pool_tok = torch.from_numpy(np.concatenate(pool_tok)).to(dev)
        Kd[:, pool_tok] = Kfull
        Vd[:, pool_tok] = Vfull

    return LayerInputs(layer=layer, tokUK=tokUK, SK=SK, VtK=VtK, tokUV=tokUV, SV=SV, VtV=VtV,
                       rank_k=rank_k, rank_v=rank_v, Kfull=Kfull, Vfull=Vfull,
                       W=make_routing_weights(spec, layer, dev), K=Kd, V=Vd)


# --------------------------------------------------------------------------------------------
# Queries
# --------------------------------------------------------------------------------------------
def make_queries(spec: WorkloadSpec, step: int = 0, device="cpu") -> torch.Tensor:
    """q ~ N(0,1), [L, B, H_q, d_h] in the storage dtype, per decode step."""
    g = _gen(device, spec.seed, 0x0E27, step)
    q = torch.randn((spec.n_layers, spec.batch, spec.n_q_heads, spec.head_dim), generator=g,
                    device=device, dtype=torch.float32)
    return q.to(storage_torch_dtype(spec.dtype))


def next_queries_ar1(spec: WorkloadSpec, q_prev: torch.Tensor, step: int, rho: float) -> torch.Tensor:
    """AR(1) query stream q_{t+1} = rho q_t + sqrt(1-rho^2) eps: rho sets how much
    consecutive steps' zoom sets overlap, i.e. the device factor-cache hit rate."""
    eps = make_queries(spec, step, q_prev.device).to(torch.float32)
    q = rho * q_prev.to(torch.float32) + (1.0 - rho * rho) ** 0.5 * eps
    return q.to(q_prev.dtype)
