"""sekv_segment_counts_static (include/sekv.h): the segmentation counts on scratch held in a static device array --
an entry point that allocates nothing -- against the existing path (sekv_build_sizes with H, which takes the same
scratch from a temporary cudaMalloc).  Integer outputs: bit-exact, like every index comparison in these tests.
The file name keeps it last in pytest's collection order."""
from __future__ import annotations

import numpy as np
import pytest
import torch

from workloads import get_spec, make_layouts

pytestmark = pytest.mark.gpu

DEV = "cuda:0"


def _batch(spec):
    from paper_2606_31145_b200 import binding as B
    from paper_2606_31145_b200 import engine as E
    lay = make_layouts(spec)
    cfg = B.make_config(n_layers=spec.n_layers, n_q_heads=spec.n_q_heads, n_kv_heads=spec.n_kv_heads,
                        head_dim=spec.head_dim, route_dim=spec.route_dim, dtype=B.SEKV_BF16, out_dtype=B.SEKV_BF16,
                        alpha=spec.alpha, l_min=spec.l_min, r_max=spec.rank, window=spec.window, max_seqs=len(lay))
    return cfg, E.seq_tok_off(lay), E.surprisal_device(lay, DEV), lay


def _existing(cfg, off, H):
    from paper_2606_31145_b200 import binding as B
    _, spans, pool = B.sekv_build_sizes(cfg, off, H)
    return np.stack([np.asarray(pool), np.asarray(spans)], axis=1).astype(np.int32)


def test_static_scratch_counts_match_build_sizes_on_two_calls_in_a_row():
    from paper_2606_31145_b200 import binding as B
    # a ragged batch (8 sequences, 8K..64K tokens), then a DIFFERENT, smaller one: the second call runs over the
    # first call's leftovers in the shared array; then the first again.  One output buffer per call.
    big = _batch(get_spec(3, batch=8))
    small = _batch(get_spec(3, case=1, batch=3, window=300))
    calls = [big, small, big]
    outs = [torch.full((len(c[1]) - 1, 2), -7, dtype=torch.int32, device=DEV) for c in calls]
    flags = [torch.full((1,), -7, dtype=torch.int32, device=DEV) for _ in calls]
    for (cfg, off, H, _), o, f in zip(calls, outs, flags):          # back to back on one stream, no sync between
        B.sekv_segment_counts_static(cfg, off, H, o, f)
    torch.cuda.synchronize()
    for (cfg, off, H, lay), o, f in zip(calls, outs, flags):
        want = _existing(cfg, off, H)
        got = o.cpu().numpy()
        assert int(f.item()) == 0
        assert np.array_equal(got, want), (got, want)
        assert (got[:, 1] > 0).all() and int(got.sum()) < off[-1]   # (not a vacuous comparison)
        if cfg.window == 0:                                          # the generator's planted layout, as a cross-check
            assert np.array_equal(got[:, 0], np.asarray([l.A for l in lay]))
            assert np.array_equal(got[:, 1], np.asarray([l.m for l in lay]))


def test_static_scratch_reports_runs_longer_than_the_span_limit():
    from paper_2606_31145_b200 import binding as B
    cfg, off, H, _ = _batch(get_spec(0))
    flat = torch.ones_like(H)                                       # constant surprisal: one run of 4096 > 1024 tokens
    o = torch.zeros((1, 2), dtype=torch.int32, device=DEV)
    f = torch.zeros((1,), dtype=torch.int32, device=DEV)
    B.sekv_segment_counts_static(cfg, off, flat, o, f)
    torch.cuda.synchronize()
    assert int(f.item()) == 1
    with pytest.raises(B.SekvError) as ei:                          # the existing path says UNSUPPORTED there
        B.sekv_build_sizes(cfg, off, flat)
    assert ei.value.status == B.SEKV_UNSUPPORTED
    B.sekv_segment_counts_static(cfg, off, H, o, f)                 # and the flag does not stick
    torch.cuda.synchronize()
    assert int(f.item()) == 0 and np.array_equal(o.cpu().numpy(), _existing(cfg, off, H))


def test_static_scratch_rejects_sizes_beyond_its_maximum():
    from paper_2606_31145_b200 import binding as B
    cfg, off, H, _ = _batch(get_spec(0))
    o = torch.full((1, 2), -7, dtype=torch.int32, device=DEV)
    f = torch.full((1,), -7, dtype=torch.int32, device=DEV)
    with pytest.raises(B.SekvError) as ei:
        B.sekv_segment_counts_static(cfg, [0, B.SEKV_STATIC_MAX_TOKENS + 1], H, o, f)
    assert ei.value.status == B.SEKV_UNSUPPORTED and "SEKV_STATIC_MAX_TOKENS" in str(ei.value)
    many = list(range(B.SEKV_STATIC_MAX_SEQS + 2))
    o2 = torch.full((len(many) - 1, 2), -7, dtype=torch.int32, device=DEV)
    with pytest.raises(B.SekvError) as ei:
        B.sekv_segment_counts_static(cfg, many, H, o2, f)
    assert ei.value.status == B.SEKV_UNSUPPORTED and "SEKV_STATIC_MAX_SEQS" in str(ei.value)
    torch.cuda.synchronize()
    assert int(o.min().item()) == -7 and int(f.item()) == -7       # nothing was launched, outputs untouched
