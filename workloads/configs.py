"""The five workload configurations of BASELINE.json (``configs[0..4]``), as data.

Every number here is quoted from BASELINE.json ``configs`` or SURVEY.md section 8(d); the paper's
hyper-parameters are cited where they come from PAPER.md (alpha = 1.0, L_min = 16, d' = 32:
PAPER.md L176 / L348; model shape 32 q heads / 8 kv heads / d_h = 128: PAPER.md L158-160).
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Tuple

import numpy as np

SEED_BASE = 0x5EC0_0000


def seed_for(config_id: int, case: int = 0) -> int:
    """seed = 0x5EC0_0000 + 1000*config + case."""
    return SEED_BASE + 1000 * int(config_id) + int(case)


@dataclass(frozen=True)
class WorkloadSpec:
    name: str
    config_id: int
    case: int
    n_layers: int
    n_q_heads: int
    n_kv_heads: int
    contexts: Tuple[int, ...]          # tokens per sequence (len = batch)
    dtype: str                         # storage dtype: "f32" | "bf16"
    rank: int                          # r (same for K and V, clipped to |S|)
    top_k: int                         # zoom cap per KV head; -1 = all spans
    len_lo: int
    len_hi: int
    anchors_per_span: int
    head_dim: int = 128
    route_dim: int = 32                # d'
    l_min: int = 16
    alpha: float = 1.0
    window: int = 0                    # configs use no local window (SURVEY reading #21)
    # "sharp sibling" scales (SURVEY.md 8(c) test-sensitivity warning); 1.0 = configs as written
    scale_sk: float = 1.0              # singular values of span keys
    scale_sv: float = 1.0              # singular values of span values
    scale_anchor_k: float = 1.0        # full-resolution (anchor) keys
    scale_w: float = 1.0               # routing projection
    notes: str = ""

    @property
    def batch(self) -> int:
        return len(self.contexts)

    @property
    def group(self) -> int:
        return self.n_q_heads // self.n_kv_heads

    @property
    def seed(self) -> int:
        return seed_for(self.config_id, self.case)

    def sharp(self) -> "WorkloadSpec":
        """Same seed, singular values / anchors / W rescaled so that token logits have std ~ 2 and the
        routing query term std ~ 1.5; calibration recorded here as constants."""
        return replace(self, name=self.name + "-sharp", scale_sk=200.0, scale_sv=20.0,
                       scale_anchor_k=16.0, scale_w=8.0)

    def with_(self, **kw) -> "WorkloadSpec":
        return replace(self, **kw)


def _ragged_contexts(config_id: int, case: int, batch: int, lo: int, hi: int) -> Tuple[int, ...]:
    rng = np.random.Generator(np.random.PCG64(seed_for(config_id, case) ^ 0xC0FFEE))
    return tuple(int(x) for x in rng.integers(lo, hi + 1, size=batch))


def get_spec(config_id: int, case: int = 0, **kw) -> WorkloadSpec:
    """Return configs[config_id].  Keyword overrides:
    config 3: batch=<1..64>; config 4: rank=<4..64>, top_k=<0|8|64|-1>; any: n_layers, contexts."""
    if config_id == 0:
        spec = WorkloadSpec("cfg0-tiny-4k-f32", 0, case, n_layers=1, n_q_heads=4, n_kv_heads=1,
                            contexts=(4096,), dtype="f32", rank=8, top_k=4, len_lo=32, len_hi=128,
                            anchors_per_span=2)
    elif config_id == 1:
        spec = WorkloadSpec("cfg1-llama8b-32k", 1, case, n_layers=1, n_q_heads=32, n_kv_heads=8,
                            contexts=(32768,), dtype="bf16", rank=16, top_k=16, len_lo=16, len_hi=256,
                            anchors_per_span=4)
    elif config_id == 2:
        spec = WorkloadSpec("cfg2-llama8b-128k-b4-L32", 2, case, n_layers=32, n_q_heads=32, n_kv_heads=8,
                            contexts=(131072,) * 4, dtype="bf16", rank=16, top_k=32, len_lo=16, len_hi=256,
                            anchors_per_span=4)
    elif config_id == 3:
        batch = int(kw.pop("batch", 8))
        spec = WorkloadSpec(f"cfg3-ragged-b{batch}", 3, case, n_layers=1, n_q_heads=32, n_kv_heads=8,
                            contexts=_ragged_contexts(3, case, batch, 8192, 65536), dtype="bf16", rank=16,
                            top_k=16, len_lo=16, len_hi=256, anchors_per_span=4)
    elif config_id == 4:
        rank = int(kw.pop("rank", 16))
        top_k = int(kw.pop("top_k", 8))
        spec = WorkloadSpec(f"cfg4-stress-64k-r{rank}-k{top_k}", 4, case, n_layers=1, n_q_heads=28,
                            n_kv_heads=4, contexts=(65536,), dtype="bf16", rank=rank, top_k=top_k,
                            len_lo=16, len_hi=256, anchors_per_span=4)
    else:
        raise ValueError(f"unknown config {config_id}")
    if kw:
        spec = replace(spec, **kw)
    return spec


CONFIGS = tuple(range(5))
