"""SeKV oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

A plain, slow, CPU, fp64 restatement of what the SeKV decode hot path computes, written from
PAPER.md (arxiv/paper_2606_31145) step by step in the paper's order and notation.  It exists to
check the CUDA library in ``paper_2606_31145_b200/``; it shares no code with it and is imported
only by ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl
reference`` legs.  Nothing in the product path may import this module.

The method is an approximation of dense attention, so the oracle follows the
algorithm: segmentation (sec. 3.1), dual-resolution representation (sec. 3.2), zoom-in routing and
mixed-resolution attention (sec. 3.3).  Floating point is fp64 on the *stored* inputs (bf16 or
fp32 values up-cast exactly).  There is no blocking, fusion or reordering: zoomed spans are
materialised explicitly as ``U diag(sigma) V^T`` (Eq. 8) and one softmax runs over all entries.

Readings of the paper where it is silent or ambiguous are those of SURVEY.md 8(c) / DESIGN.md
section 3 and are flagged ``[reading #n]`` below.

Pins (tests/test_oracle_*.py, ``-m "not gpu"``): every function here is pinned against something
other than itself -- the paper's printed numbers, closed forms, LAPACK, torch's dense
scaled-dot-product attention, brute force -- see DESIGN.md section 5.  Unpinned: nothing in this
file; the paper's *trained* W / tau / g_phi and its accuracy tables are "parity unpinned" because
weights and datasets do not exist here (synthetic stand-ins only).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np


# =============================================================================================
# Storage rounding
# =============================================================================================
def round_bf16(x: np.ndarray) -> np.ndarray:
    """Round to bfloat16 (round-to-nearest-even on the upper 16 bits of the fp32 pattern) and
    return the values as float64.  bf16 is the storage dtype of configs 1-4 (BASELINE.json)."""
    f = np.ascontiguousarray(np.asarray(x, dtype=np.float32))
    u = f.view(np.uint32).astype(np.uint64)
    lsb = (u >> 16) & 1
    r = ((u + 0x7FFF + lsb) >> 16) << 16
    out = r.astype(np.uint32).view(np.float32)
    out = np.where(np.isfinite(f), out, f)
    return out.astype(np.float64).reshape(np.shape(x))


def round_storage(x: np.ndarray, dtype: str) -> np.ndarray:
    if dtype == "bf16":
        return round_bf16(x)
    if dtype == "f32":
        return np.asarray(x, dtype=np.float32).astype(np.float64)
    raise ValueError(dtype)


# =============================================================================================
# 3.1  Entropy-guided span segmentation
# =============================================================================================
def surprisal_threshold(H: np.ndarray, alpha: float) -> float:
    """mu + alpha*sigma over the sequence.  [reading #1] sigma is the population
    standard deviation (ddof = 0)."""
    H = np.asarray(H, dtype=np.float64)
    mu = H.sum() / H.shape[0]
    sigma = np.sqrt(((H - mu) ** 2).sum() / H.shape[0])
    return float(mu + alpha * sigma)


@dataclass
class Segmentation:
    n: int
    pool_pos: np.ndarray      # [A] positions kept at full resolution (anchors, short runs, window)
    span_start: np.ndarray    # [m]
    span_len: np.ndarray      # [m]

    @property
    def m(self) -> int:
        return int(self.span_len.shape[0])

    @property
    def A(self) -> int:
        return int(self.pool_pos.shape[0])


def segment(H: np.ndarray, alpha: float = 1.0, l_min: int = 16, window: int = 0) -> Segmentation:
    """positions with H_t > mu + alpha*sigma are span boundaries, retained as anchor
    tokens at full resolution; the tokens between two neighbouring anchors form a span.
    [reading #2] strict '>'.  [reading #3] leading / trailing runs are spans too.
    [reading #4] adjacent boundary tokens are each an anchor; there are no empty spans.
    [reading #5] PAPER.md L108: runs shorter than L_min stay at full resolution (join the pool).
    [reading #21] Eq. 17: the last ``window`` tokens are full resolution."""
    H = np.asarray(H, dtype=np.float64)
    n = int(H.shape[0])
    thr = surprisal_threshold(H, alpha)
    full = H > thr
    if window > 0:
        full[max(0, n - window):] = True
    starts: List[int] = []
    lens: List[int] = []
    t = 0
    while t < n:
        if full[t]:
            t += 1
            continue
        s = t
        while t < n and not full[t]:
            t += 1
        if t - s < l_min:
            full[s:t] = True
        else:
            starts.append(s)
            lens.append(t - s)
    return Segmentation(n=n, pool_pos=np.nonzero(full)[0].astype(np.int64),
                        span_start=np.asarray(starts, dtype=np.int64),
                        span_len=np.asarray(lens, dtype=np.int64))


# =============================================================================================
# 3.2  Dual-resolution span representation
# =============================================================================================
def span_weights(H_span: np.ndarray) -> np.ndarray:
    """Eq. 2: w_t = H_t / sum_{k in S} H_k.  [reading #6] uniform if the sum is zero."""
    H_span = np.asarray(H_span, dtype=np.float64)
    tot = H_span.sum()
    if tot == 0.0:
        return np.full(H_span.shape[0], 1.0 / H_span.shape[0])
    return H_span / tot


def coarse_mean(w: np.ndarray, X_span: np.ndarray) -> np.ndarray:
    """k_bar_S = sum_t w_t K_t (same for v_bar_S with V)."""
    return np.asarray(w, dtype=np.float64) @ np.asarray(X_span, dtype=np.float64)


def routing_summary(w: np.ndarray, K_span: np.ndarray, W_h: np.ndarray) -> np.ndarray:
    """Eq. 3: K_bar_S = normalize_2( sum_t w_t W K_t ) in R^{d'}; one per query head, built from
    its group's shared kv head."""
    WK = np.asarray(K_span, dtype=np.float64) @ np.asarray(W_h, dtype=np.float64).T   # row t = W K_t
    acc = np.asarray(w, dtype=np.float64) @ WK                                        # sum_t w_t W K_t
    nrm = np.sqrt((acc * acc).sum())
    if nrm == 0.0:
        return acc
    return acc / nrm


def truncated_svd(X_span: np.ndarray, r_max: int) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Eq. 6: K_S = sum_{i<=R} sigma_i u_i v_i^T with R = min(|S|, d_h, R_max).  The SVD itself is
    LAPACK's (numpy.linalg.svd), a textbook routine.  Returns U [|S|,R], sigma [R], Vt [R,d_h]."""
    U, s, Vt = np.linalg.svd(np.asarray(X_span, dtype=np.float64), full_matrices=False)
    R = int(min(X_span.shape[0], X_span.shape[1], r_max))
    return U[:, :R].copy(), s[:R].copy(), Vt[:R].copy()


def gated_reconstruction(U: np.ndarray, sigma: np.ndarray, Vt: np.ndarray,
                         gates: Optional[np.ndarray] = None) -> np.ndarray:
    """Eq. 8: K_hat_S = sum_i m_i sigma_i u_i v_i^T.  [reading #19] at deployment the gates are
    binary and the stored factors are the kept components, so ``gates=None`` means all ones."""
    R = sigma.shape[0]
    m = np.ones(R) if gates is None else np.asarray(gates, dtype=np.float64)
    out = np.zeros((U.shape[0], Vt.shape[1]), dtype=np.float64)
    for i in range(R):
        out += (m[i] * sigma[i]) * np.outer(U[:, i], Vt[i])
    return out


def gated_error(gates: np.ndarray, sigma_all: np.ndarray) -> float:
    """E(m, sigma) = sum_i (1 - m_i)^2 sigma_i^2."""
    gates = np.asarray(gates, dtype=np.float64)
    sigma_all = np.asarray(sigma_all, dtype=np.float64)
    return float((((1.0 - gates) ** 2) * sigma_all ** 2).sum())


@dataclass
class SpanFactors:
    """Stored low-rank factors of one (kv head, span): the paper's U_S, Sigma_S (as r values,
    [reading #20]), V_S for keys and for values."""
    UK: np.ndarray
    sK: np.ndarray
    VtK: np.ndarray
    UV: np.ndarray
    sV: np.ndarray
    VtV: np.ndarray


@dataclass
class Tables:
    """The stored hierarchical memory of ONE sequence at ONE layer:
    GPU side: full-resolution pool K/V, coarse means, routing summaries; CPU side: factors."""
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    route_dim: int
    seg: Segmentation
    full_K: np.ndarray     # [H_kv, A, d_h]
    full_V: np.ndarray
    mean_K: np.ndarray     # [H_kv, m, d_h]   k_bar_S
    mean_V: np.ndarray     # [H_kv, m, d_h]   v_bar_S
    route_K: np.ndarray    # [H_q, m, d']     K_bar_S
    W: np.ndarray          # [H_q, d', d_h]
    factors: List[List[SpanFactors]] = field(default_factory=list)   # [H_kv][m]

    @property
    def group(self) -> int:
        return self.n_q_heads // self.n_kv_heads


def build_tables(H: np.ndarray, K: np.ndarray, V: np.ndarray, W: np.ndarray, *, alpha: float = 1.0,
                 l_min: int = 16, r_max: int = 32, window: int = 0, dtype: str = "bf16",
                 prefactored: Optional[Dict[str, np.ndarray]] = None) -> Tables:
    """Prefill-time construction for one sequence at one layer (sec. 3.1-3.2).

    ``K, V`` [H_kv, n, d_h] and ``W`` [H_q, d', d_h] hold stored (already quantised) values.
    Results that the method stores (k_bar, v_bar, K_bar, U, V^T) are rounded to the storage dtype;
    sigma stays fp32 [reading #20].

    ``prefactored``: the generator's own factors for the *planted* spans (tokU* [H_kv, n, r],
    S* [H_kv, m, r], Vt* [H_kv, m, r, d_h], rank_* [H_kv, m]); then K, V may hold only the pool
    tokens' rows, the span rows of K/V are DEFINED as U diag(S) V^T (materialised here), and the
    stored factors are the given ones (the SVD of Eq. 6 is skipped)."""
    H = np.asarray(H, dtype=np.float64)
    hk, n, d = K.shape
    hq, dp, _ = W.shape
    G = hq // hk
    seg = segment(H, alpha, l_min, window)
    m, A = seg.m, seg.A
    full_K = np.asarray(K[:, seg.pool_pos, :], dtype=np.float64)
    full_V = np.asarray(V[:, seg.pool_pos, :], dtype=np.float64)
    mean_K = np.zeros((hk, m, d))
    mean_V = np.zeros((hk, m, d))
    route_K = np.zeros((hq, m, dp))
    factors: List[List[SpanFactors]] = [[None] * m for _ in range(hk)]  # type: ignore
    for s in range(m):
        a, ln = int(seg.span_start[s]), int(seg.span_len[s])
        w = span_weights(H[a:a + ln])
        for g in range(hk):
            if prefactored is not None:
                rk = int(prefactored["rank_k"][g, s])
                rv = int(prefactored["rank_v"][g, s])
                f = SpanFactors(
                    UK=np.asarray(prefactored["tokUK"][g, a:a + ln, :rk], dtype=np.float64),
                    sK=np.asarray(prefactored["SK"][g, s, :rk], dtype=np.float64),
                    VtK=np.asarray(prefactored["VtK"][g, s, :rk, :], dtype=np.float64),
                    UV=np.asarray(prefactored["tokUV"][g, a:a + ln, :rv], dtype=np.float64),
                    sV=np.asarray(prefactored["SV"][g, s, :rv], dtype=np.float64),
                    VtV=np.asarray(prefactored["VtV"][g, s, :rv, :], dtype=np.float64))
                K_S = gated_reconstruction(f.UK, f.sK, f.VtK)
                V_S = gated_reconstruction(f.UV, f.sV, f.VtV)
            else:
                K_S = np.asarray(K[g, a:a + ln, :], dtype=np.float64)
                V_S = np.asarray(V[g, a:a + ln, :], dtype=np.float64)
                UK, sK, VtK = truncated_svd(K_S, r_max)
                UV, sV, VtV = truncated_svd(V_S, r_max)
                f = SpanFactors(UK=round_storage(UK, dtype), sK=round_storage(sK, "f32"),
                                VtK=round_storage(VtK, dtype), UV=round_storage(UV, dtype),
                                sV=round_storage(sV, "f32"), VtV=round_storage(VtV, dtype))
            factors[g][s] = f
            mean_K[g, s] = coarse_mean(w, K_S)
            mean_V[g, s] = coarse_mean(w, V_S)
            for h in range(g * G, (g + 1) * G):
                route_K[h, s] = routing_summary(w, K_S, np.asarray(W[h], dtype=np.float64))
    return Tables(n_q_heads=hq, n_kv_heads=hk, head_dim=d, route_dim=dp, seg=seg,
                  full_K=full_K, full_V=full_V,
                  mean_K=round_storage(mean_K, dtype), mean_V=round_storage(mean_V, dtype),
                  route_K=round_storage(route_K, dtype), W=np.asarray(W, dtype=np.float64),
                  factors=factors)


# =============================================================================================
# 3.3  Zoom-in routing
# =============================================================================================
def sigmoid(x: np.ndarray) -> np.ndarray:
    """sig(x) = 1 / (1 + e^{-x})."""
    return 1.0 / (1.0 + np.exp(-np.asarray(x, dtype=np.float64)))


@dataclass
class RouteResult:
    logit: np.ndarray      # x [H_q, m]: the argument of the sigmoid in Eq. 5
    alpha: np.ndarray      # alpha_tilde [H_q, m]
    group_logit: np.ndarray  # X [H_kv, m] = max over the group's query heads  [reading #10]
    ids: List[np.ndarray]  # per kv head: zoomed span ids in decreasing-score order


def route(q: np.ndarray, W: np.ndarray, route_K: np.ndarray, span_len: np.ndarray, n_kv_heads: int,
          k: int, tau: Optional[np.ndarray] = None) -> RouteResult:
    """Eq. 4: q' = W q.  Eq. 5: alpha_tilde = sig(q' . K_bar / sqrt(d') + log|S|)  [reading #14:
    natural log].  Eq. 9: z = 1[alpha_tilde > tau].  PAPER.md L123: under a budget keep spans in
    decreasing alpha_tilde order until it is filled.
    [reading #9] ranking uses the pre-sigmoid logit x (same order as alpha_tilde, no saturation).
    [reading #10] selection is per KV head: X_{g,s} = max_{h in g} x_{h,s}; a span is eligible if
    any head of the group passes its threshold.  [reading #12/#13] the budget is k spans per
    (sequence, layer, kv head); k < 0 means no cap.  Ties go to the lower span id."""
    q = np.asarray(q, dtype=np.float64)
    hq, dp, d = W.shape
    m = int(span_len.shape[0])
    G = hq // n_kv_heads
    x = np.zeros((hq, m))
    for h in range(hq):
        qp = np.asarray(W[h], dtype=np.float64) @ q[h]                  # Eq. 4
        if m:
            x[h] = (np.asarray(route_K[h], dtype=np.float64) @ qp) / np.sqrt(dp) \
                + np.log(np.asarray(span_len, dtype=np.float64))                       # Eq. 5
    alpha = sigmoid(x)
    X = np.zeros((n_kv_heads, m))
    ids: List[np.ndarray] = []
    for g in range(n_kv_heads):
        hs = range(g * G, (g + 1) * G)
        X[g] = x[list(hs)].max(axis=0) if m else np.zeros(0)
        if tau is None:
            eligible = np.ones(m, dtype=bool)
        else:
            eligible = np.zeros(m, dtype=bool)
            for h in hs:
                eligible |= alpha[h] > float(tau[h])                    # Eq. 9
        cand = [s for s in range(m) if eligible[s]]
        cand.sort(key=lambda s: (-X[g, s], s))                          # decreasing score, ties -> lower id
        cap = len(cand) if k < 0 else min(k, len(cand))
        ids.append(np.asarray(cand[:cap], dtype=np.int64))
    return RouteResult(logit=x, alpha=alpha, group_logit=X, ids=ids)


# =============================================================================================
# 3.3  Mixed-resolution attention
# =============================================================================================
def softmax_attend(logits: np.ndarray, values: np.ndarray) -> Tuple[np.ndarray, float]:
    """One max-subtracted softmax over all entries and the weighted sum of their values.
    Returns (out, log-sum-exp).  An empty entry list gives (0, -inf)."""
    if logits.shape[0] == 0:
        return np.zeros(values.shape[1]), float("-inf")
    mx = logits.max()
    if not np.isfinite(mx):
        return np.zeros(values.shape[1]), float("-inf")
    p = np.exp(logits - mx)
    l = p.sum()
    out = (p[:, None] * values).sum(axis=0) / l
    return out, float(mx + np.log(l))


def mixed_entries(q_h: np.ndarray, g: int, T: Tables, zoom: Sequence[int]) -> Tuple[np.ndarray, np.ndarray]:
    """The entry list of PAPER.md L119-121 for one query head whose kv head is g:
    anchors/pool tokens with their full key-value pairs; one coarse entry (k_bar, v_bar) with a
    +log|S| score correction per NON-expanded span; the reconstructed tokens (Eq. 8) of every
    expanded span.  [reading #15] score scale 1/sqrt(d_h).  [reading #17] an expanded span's
    coarse entry is replaced by its tokens ("zooming refines ... no span is dropped", L121)."""
    d = T.head_dim
    scale = 1.0 / np.sqrt(d)
    zoomset = set(int(s) for s in zoom)
    logits: List[np.ndarray] = []
    values: List[np.ndarray] = []
    if T.seg.A:
        logits.append((T.full_K[g] @ q_h) * scale)
        values.append(T.full_V[g])
    for s in range(T.seg.m):
        if s in zoomset:
            f = T.factors[g][s]
            K_hat = gated_reconstruction(f.UK, f.sK, f.VtK)            # Eq. 8, materialised
            V_hat = gated_reconstruction(f.UV, f.sV, f.VtV)
            logits.append((K_hat @ q_h) * scale)
            values.append(V_hat)
        else:
            logits.append(np.asarray([(T.mean_K[g, s] @ q_h) * scale + np.log(float(T.seg.span_len[s]))]))
            values.append(T.mean_V[g, s][None, :])
    if not logits:
        return np.zeros(0), np.zeros((0, d))
    return np.concatenate(logits), np.concatenate(values, axis=0)


def decode_attn(q: np.ndarray, T: Tables, zoom_ids: Sequence[Sequence[int]],
                heads: Optional[Sequence[int]] = None) -> Tuple[np.ndarray, np.ndarray]:
    """Mixed-resolution attention for every query head of one sequence at one layer.
    ``q`` [H_q, d_h]; ``zoom_ids[g]`` the expanded spans of kv head g.  Returns out [H_q, d_h] and
    the log-sum-exp [H_q] of each head's softmax.  ``heads`` restricts the work to a subset of
    query heads (the other rows stay zero) so that tests can sample large configurations."""
    q = np.asarray(q, dtype=np.float64)
    G = T.group
    out = np.zeros((T.n_q_heads, T.head_dim))
    lse = np.zeros(T.n_q_heads)
    for h in (range(T.n_q_heads) if heads is None else heads):
        g = h // G
        logits, values = mixed_entries(q[h], g, T, zoom_ids[g])
        out[h], lse[h] = softmax_attend(logits, values)
    return out, lse


def merge_partials(parts: Sequence[Tuple[np.ndarray, float]]) -> Tuple[np.ndarray, float]:
    """PAPER.md L61 "outputs merged across both stages" [reading #18]: partial softmax results
    (normalised out_i, lse_i) over disjoint entry sets merge to the result over their union:
    lse = log sum_i e^{lse_i},  out = sum_i e^{lse_i - lse} out_i."""
    lses = np.asarray([p[1] for p in parts], dtype=np.float64)
    mx = lses.max()
    if not np.isfinite(mx):
        return np.zeros_like(parts[0][0]), float("-inf")
    wts = np.exp(lses - mx)
    tot = wts.sum()
    out = sum(w * p[0] for w, p in zip(wts, parts)) / tot
    return out, float(mx + np.log(tot))


# =============================================================================================
# Appendix D  byte accounting
# =============================================================================================
def fullkv_bytes(L: int, H_kv: int, d_h: int, n: int, b: int) -> int:
    """Eq. 16: Mem_FullKV = 2 L H_kv d_h n b."""
    return 2 * L * H_kv * d_h * n * b


def sekv_gpu_bytes(L: int, H_kv: int, H: int, d_h: int, d_route: int, a: int, w: int, m: int, b: int) -> int:
    """Eq. 17: Mem_GPU ~= 2 L H_kv d_h (a + w) b + 2 L H d' m b."""
    return 2 * L * H_kv * d_h * (a + w) * b + 2 * L * H * d_route * m * b


def sekv_cpu_span_values(r: int, span_len: int, d_h: int) -> int:
    """a retained rank-r factorisation costs r(|S| + d_h + 1) values."""
    return r * (span_len + d_h + 1)


def sekv_cpu_span_bytes(L: int, H_kv: int, r: int, span_len: int, d_h: int, b: int) -> int:
    """Eq. 18: Mem_CPU(S) = 2 L H_kv r (|S| + d_h + 1) b (keys and values)."""
    return 2 * L * H_kv * sekv_cpu_span_values(r, span_len, d_h) * b


def transfer_bytes(L: int, H_kv: int, r: int, zoom_lens: Sequence[int], d_h: int, b: int) -> int:
    """Eq. 20: Transfer_t = sum_{S in Z_t} 2 L H_kv r (|S| + d_h + 1) b."""
    return sum(sekv_cpu_span_bytes(L, H_kv, r, int(s), d_h, b) for s in zoom_lens)


def routing_parameters(L: int, H: int, d_route: int, d_h: int) -> int:
    """{W^(l,h)} in R^{L x H x d' x d_h}."""
    return L * H * d_route * d_h
