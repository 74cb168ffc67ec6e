"""Test-side glue: read golden fixtures, hand generator tensors to the oracle as numpy arrays."""
from __future__ import annotations

import os
from typing import Dict, List, Sequence

import numpy as np
import torch

from oracle import sekv_oracle as O
from workloads import LayerInputs, SequenceLayout, WorkloadSpec

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_golden(name: str) -> Dict[str, List[float]]:
    out: Dict[str, List[float]] = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line or "=" not in line:
                continue
            k, v = line.split("=", 1)
            out[k.strip()] = [float(x) for x in v.split()]
    return out


def to_np(t: torch.Tensor) -> np.ndarray:
    """Exact up-cast of a stored tensor (bf16 / fp32 / int) to float64 / int64 numpy."""
    t = t.detach().cpu()
    if t.dtype in (torch.bfloat16, torch.float16, torch.float32):
        return t.to(torch.float32).numpy().astype(np.float64)
    if t.dtype == torch.float64:
        return t.numpy()
    return t.numpy().astype(np.int64)


def seq_offsets(layouts: Sequence[SequenceLayout]):
    tok = np.zeros(len(layouts) + 1, dtype=np.int64)
    spn = np.zeros(len(layouts) + 1, dtype=np.int64)
    pool = np.zeros(len(layouts) + 1, dtype=np.int64)
    for b, l in enumerate(layouts):
        tok[b + 1] = tok[b] + l.n
        spn[b + 1] = spn[b] + l.m
        pool[b + 1] = pool[b] + l.A
    return tok, spn, pool


def oracle_tables(spec: WorkloadSpec, layouts: Sequence[SequenceLayout], li: LayerInputs, b: int,
                  mode: str = "prefactored", r_max: int | None = None) -> O.Tables:
    """Run the oracle's prefill-time construction (steps 1-3) for sequence ``b`` of a layer."""
    tok, spn, pool = seq_offsets(layouts)
    l = layouts[b]
    t0, t1 = int(tok[b]), int(tok[b + 1])
    s0, s1 = int(spn[b]), int(spn[b + 1])
    p0, p1 = int(pool[b]), int(pool[b + 1])
    W = to_np(li.W)
    if mode == "dense":
        assert li.K is not None
        return O.build_tables(l.H, to_np(li.K[:, t0:t1]), to_np(li.V[:, t0:t1]), W, alpha=spec.alpha,
                              l_min=spec.l_min, r_max=r_max or spec.rank, window=spec.window,
                              dtype=spec.dtype)
    hk, d = spec.n_kv_heads, spec.head_dim
    K = np.zeros((hk, l.n, d))
    V = np.zeros((hk, l.n, d))
    K[:, l.planted_pool_pos] = to_np(li.Kfull[:, p0:p1])
    V[:, l.planted_pool_pos] = to_np(li.Vfull[:, p0:p1])
    pre = dict(tokUK=to_np(li.tokUK[:, t0:t1]), SK=to_np(li.SK[:, s0:s1]), VtK=to_np(li.VtK[:, s0:s1]),
               tokUV=to_np(li.tokUV[:, t0:t1]), SV=to_np(li.SV[:, s0:s1]), VtV=to_np(li.VtV[:, s0:s1]),
               rank_k=to_np(li.rank_k[:, s0:s1]), rank_v=to_np(li.rank_v[:, s0:s1]))
    T = O.build_tables(l.H, K, V, W, alpha=spec.alpha, l_min=spec.l_min, r_max=spec.rank,
                       window=spec.window, dtype=spec.dtype, prefactored=pre)
    assert np.array_equal(T.seg.span_start, l.planted_span_start), "segmentation != planted layout"
    assert np.array_equal(T.seg.span_len, l.planted_span_len)
    assert np.array_equal(T.seg.pool_pos, l.planted_pool_pos)
    return T


def rel_l2(a: np.ndarray, b: np.ndarray) -> float:
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    den = np.sqrt((b * b).sum())
    return float(np.sqrt(((a - b) ** 2).sum()) / (den if den > 0 else 1.0))


def check_ids(got: Sequence[int], ref: Sequence[int], ref_score: np.ndarray, gap: float = 1e-4) -> None:
    """BASELINE.json: routing indices bit-exact, ties broken by lower span id, or compared as sets
    where the score gap is below 1e-4.  Position by position the ids must match, or the two spans'
    oracle scores must differ by less than ``gap``; as sets they must match except for swaps across
    the cut between spans whose scores are within ``gap`` of the cut score."""
    got = [int(x) for x in got]
    ref = [int(x) for x in ref]
    assert len(got) == len(ref), (len(got), len(ref))
    for g, r in zip(got, ref):
        if g != r:
            assert abs(ref_score[g] - ref_score[r]) < gap, (g, r, ref_score[g], ref_score[r])
    assert len(set(got)) == len(got)
    if ref:
        cut = ref_score[ref[-1]]
        for g in set(got) - set(ref):
            assert abs(ref_score[g] - cut) < gap, (g, ref_score[g], cut)
