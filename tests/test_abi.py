"""CPU-only checks of the boundary: the shared library builds for sm_100a, loads, exports every symbol
that include/sekv.h declares, and its pure (no-GPU) entry points behave.  No compute calls."""
from __future__ import annotations

import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_2606_31145_b200.build import build_library
    build_library()
    from paper_2606_31145_b200 import binding as B
    return B


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "sekv.h")).read()
    return sorted(set(re.findall(r"^SEKV_API[^;(]*?\b(sekv_\w+)\s*\(", text, flags=re.M)))


def test_header_declares_the_named_entry_points():
    syms = _declared_symbols()
    for name in ("sekv_build_spans", "sekv_route", "sekv_decode_attn", "sekv_create", "sekv_destroy"):
        assert name in syms
    for name in ("sekv_build_sizes", "sekv_get_path", "sekv_export_span_factors"):
        assert name in syms
    assert len(syms) >= 21


def test_library_exports_every_declared_symbol(binding):
    lib = ctypes.CDLL(binding.LIB_PATH)
    for name in _declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/sekv.h but not exported"


def test_pure_entry_points(binding):
    B = binding
    assert "sm_100a" in B.sekv_version()
    assert B.lib.sekv_status_string(0) == b"SEKV_OK" and B.lib.sekv_status_string(6) == b"SEKV_STATE"
    # blob bytes: PAPER.md L108 count r(|S| + d_h + 1) for K and V, fp32 sigma, ranks and |S| padded to 16
    for dtype, es in ((B.SEKV_BF16, 2), (B.SEKV_F32, 4)):
        for ln, rk, rv in ((256, 16, 16), (100, 16, 16), (16, 4, 8), (77, 33, 64)):
            lp, kp, vp = -(-ln // 16) * 16, -(-rk // 16) * 16, -(-rv // 16) * 16
            raw = 4 * (kp + vp) + es * (128 * (kp + vp) + lp * (kp + vp))
            assert B.sekv_blob_bytes(dtype, ln, rk, rv) == -(-raw // 128) * 128
            algo = (rk + rv) * (ln + 128) * es + 4 * (rk + rv)
            assert B.sekv_blob_bytes(dtype, ln, rk, rv) >= algo
    cfg = B.make_config(n_layers=2, max_seqs=2, max_tokens_total=10000, max_spans_total=100, max_full_total=300,
                        k_cap=8, cache_ways=16, r_max=16)
    # sizes from token counts alone (no GPU): m_b <= n_b / l_min, A_b <= n_b
    sz, spans, pool = B.sekv_build_sizes(cfg, [0, 4096, 10000])
    assert not sz.exact and sz.tokens_total == 10000 and sz.full_total == 10000
    assert spans == [4096 // 16, 5904 // 16] and pool == [4096, 5904] and sz.spans_total == sum(spans)
    assert sz.max_span_len == 1024 and sz.host_bytes >= 2 * 8 * sum(spans) * B.sekv_blob_bytes(B.SEKV_BF16, 16, 16, 16)
    dev, slot = B.sekv_device_arena_bytes(cfg)
    assert slot == B.sekv_blob_bytes(B.SEKV_BF16, 256, 16, 16)
    assert dev > 2 * 2 * 8 * 16 * slot          # at least the factor cache
    # argument validation happens before any CUDA call
    for bad in (dict(head_dim=64), dict(n_q_heads=30), dict(route_dim=30), dict(r_max=65), dict(cache_ways=4),
                dict(n_q_heads=72, n_kv_heads=8), dict(max_span_len=2048), dict(dtype=7)):
        kw = dict(n_layers=2, max_seqs=2, max_tokens_total=10000, max_spans_total=100, max_full_total=300,
                  k_cap=8, cache_ways=16, r_max=16)
        kw.update(bad)
        with pytest.raises(B.SekvError) as ei:
            B.sekv_device_arena_bytes(B.make_config(**kw))
        assert ei.value.status == B.SEKV_INVALID_ARG


def test_create_without_gpu_fails_loudly(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    B = binding
    cfg = B.make_config(max_tokens_total=1000, max_spans_total=10, max_full_total=10)
    dev, _ = B.sekv_device_arena_bytes(cfg)
    buf = (ctypes.c_uint8 * 8192)()
    addr = (ctypes.addressof(buf) + 255) // 256 * 256
    h = ctypes.c_void_p(None)
    st = B.lib.sekv_create(ctypes.byref(cfg), addr, dev, addr, 4096, ctypes.byref(h))
    assert st == B.SEKV_CUDA and not h.value          # no CPU fallback


def test_product_code_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_31145_b200")
    pat = re.compile(r"^\s*(from\s+oracle|import\s+oracle|#\s*include\s+[\"<][^\">]*oracle)", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not pat.search(text), f"{f} pulls in the oracle"
                assert "sekv_oracle" not in text, f"{f} names the oracle module"
