"""Thin ctypes binding of libsekv (include/sekv.h).  Argument marshalling only: every step of the
path runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory, pinned host memory
and streams; tensors are passed as raw pointers.

There is no fallback of any kind: if the shared library is missing or fails to load, importing
this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsekv.so")

SEKV_OK, SEKV_INVALID_ARG, SEKV_UNSUPPORTED, SEKV_OOM_DEVICE, SEKV_OOM_HOST, SEKV_CUDA, SEKV_STATE = range(7)
SEKV_F32, SEKV_BF16 = 0, 1


class SekvError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        super().__init__(f"{where}: {_status_name(status)}" + (f" ({detail})" if detail else ""))


class sekv_config(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32),
                ("head_dim", C.c_int32), ("route_dim", C.c_int32), ("dtype", C.c_int32),
                ("out_dtype", C.c_int32), ("alpha", C.c_float), ("l_min", C.c_int32), ("r_max", C.c_int32),
                ("window", C.c_int32), ("max_seqs", C.c_int32), ("max_tokens_total", C.c_int64),
                ("max_spans_total", C.c_int32), ("max_full_total", C.c_int32), ("max_span_len", C.c_int32),
                ("k_cap", C.c_int32), ("cache_ways", C.c_int32), ("prefetch", C.c_int32),
                ("stage1_ctas", C.c_int32), ("item_rows", C.c_int32), ("zoom_spans_per_item", C.c_int32),
                ("use_graph", C.c_int32), ("impl", C.c_int32), ("main_stream", C.c_void_p),
                ("side_stream", C.c_void_p)]


_LAYOUT_FIELDS = ["esize", "rows_cap", "spans_cap", "seq_tok_off", "seq_row_off", "seq_span_off", "seq_pool_cnt",
                  "span_len", "span_tok_start", "ln_len", "pool_tok", "ent_k", "ent_v", "ent_layer_stride",
                  "ent_head_stride", "route", "route_layer_stride", "route_head_stride", "w", "w_layer_stride",
                  "dir_off", "dir_rank", "dir_layer_stride_elems", "cache_tags", "cache_stamps", "cache_slots",
                  "slot_bytes", "host_bytes_used", "device_bytes_total"]


class sekv_layout(C.Structure):
    _fields_ = [(n, C.c_int64) for n in _LAYOUT_FIELDS]


_STATS_FIELDS = ["layer_steps", "zoomed_spans", "cache_hits", "cache_misses", "h2d_bytes", "factor_bytes_algo",
                 "coarse_rows_skipped", "prefetched_spans", "kernel_launches", "prefetch_h2d_bytes"]


class sekv_stats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in _STATS_FIELDS]


class sekv_sizes(C.Structure):
    _fields_ = [("tokens_total", C.c_int64), ("spans_total", C.c_int32), ("full_total", C.c_int32),
                ("max_spans_per_seq", C.c_int32), ("max_span_len", C.c_int32), ("exact", C.c_int32),
                ("host_bytes", C.c_int64)]


class sekv_factors(C.Structure):
    _fields_ = [("rank_in", C.c_int32), ("tokUK", C.c_void_p), ("SK", C.c_void_p), ("VtK", C.c_void_p),
                ("tokUV", C.c_void_p), ("SV", C.c_void_p), ("VtV", C.c_void_p), ("rank_k", C.c_void_p),
                ("rank_v", C.c_void_p), ("Kfull", C.c_void_p), ("Vfull", C.c_void_p), ("a_tot", C.c_int32),
                ("m_tot", C.c_int32)]


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_31145_b200.build` "
                          "(there is no CPU or PyTorch fallback)")
    lib = C.CDLL(LIB_PATH)
    P, I32, I64, VP = C.POINTER, C.c_int32, C.c_int64, C.c_void_p
    lib.sekv_version.restype = C.c_char_p
    lib.sekv_status_string.restype = C.c_char_p
    lib.sekv_status_string.argtypes = [C.c_int]
    lib.sekv_device_arena_bytes.argtypes = [P(sekv_config), P(C.c_size_t), P(C.c_size_t)]
    lib.sekv_blob_bytes.restype = C.c_size_t
    lib.sekv_blob_bytes.argtypes = [I32, I32, I32, I32]
    lib.sekv_create.argtypes = [P(sekv_config), VP, C.c_size_t, VP, C.c_size_t, P(VP)]
    lib.sekv_destroy.restype = None
    lib.sekv_destroy.argtypes = [VP]
    lib.sekv_last_error.restype = C.c_char_p
    lib.sekv_last_error.argtypes = [VP]
    lib.sekv_build_spans.argtypes = [VP, I32, I32, P(I64), VP, VP, VP, VP, I32, P(I32), P(I32)]
    lib.sekv_build_spans_prefactored.argtypes = [VP, I32, I32, P(I64), VP, P(sekv_factors), VP, P(I32), P(I32)]
    lib.sekv_reset.argtypes = [VP]
    lib.sekv_route.argtypes = [VP, I32, VP, VP, I32, VP, VP, VP, VP]
    lib.sekv_decode_attn.argtypes = [VP, I32, VP, VP, VP, VP, VP]
    lib.sekv_decode_step.argtypes = [VP, VP, VP, I32, VP, VP]
    lib.sekv_decode_step_host.argtypes = [VP, VP, VP, I32, VP, VP]
    lib.sekv_last_zoom_ids.argtypes = [VP, I32, VP, VP]
    lib.sekv_get_layout.argtypes = [VP, P(sekv_layout)]
    lib.sekv_get_stats.argtypes = [VP, P(sekv_stats)]
    lib.sekv_reset_stats.argtypes = [VP]
    lib.sekv_cache_flush.argtypes = [VP]
    lib.sekv_static_bytes_per_layer.argtypes = [VP, P(C.c_uint64)]
    lib.sekv_get_schedule.argtypes = [VP, P(I32), P(I32)]
    lib.sekv_set_profiling.argtypes = [VP, I32]
    lib.sekv_get_kernel_times.argtypes = [VP, P(C.c_double), P(C.c_uint64)]
    lib.sekv_set_trace.argtypes = [VP, VP, I64, P(I32)]
    lib.sekv_build_sizes.argtypes = [P(sekv_config), I32, P(I64), VP, P(sekv_sizes), P(I32), P(I32)]
    lib.sekv_get_path.argtypes = [VP, P(I32), P(C.c_char_p)]
    lib.sekv_graph_count.argtypes = [VP, P(I32)]
    lib.sekv_export_span_factors.argtypes = [VP, I32, I32, I32, I32, P(I32), P(I32), P(I32), VP, VP, VP, VP, VP, VP, P(I32)]
    lib.sekv_segment_counts_static.argtypes = [P(sekv_config), I32, P(I64), VP, VP, VP, VP]
    lib.sekv_static_last_error.restype = C.c_char_p
    lib.sekv_static_last_error.argtypes = []
    for name in ("sekv_segment_counts_static", "sekv_device_arena_bytes", "sekv_create", "sekv_build_spans", "sekv_build_spans_prefactored",
                 "sekv_reset", "sekv_route", "sekv_decode_attn", "sekv_decode_step", "sekv_decode_step_host",
                 "sekv_last_zoom_ids",
                 "sekv_get_layout", "sekv_get_stats", "sekv_reset_stats", "sekv_cache_flush",
                 "sekv_static_bytes_per_layer", "sekv_get_schedule", "sekv_set_profiling",
                 "sekv_get_kernel_times", "sekv_set_trace", "sekv_build_sizes", "sekv_get_path", "sekv_graph_count",
                 "sekv_export_span_factors"):
        getattr(lib, name).restype = C.c_int
    return lib


lib = _load()


def _status_name(s: int) -> str:
    return lib.sekv_status_string(int(s)).decode()


def sekv_version() -> str:
    return lib.sekv_version().decode()


def sekv_blob_bytes(dtype: int, span_len: int, rank_k: int, rank_v: int) -> int:
    return int(lib.sekv_blob_bytes(dtype, span_len, rank_k, rank_v))


def sekv_device_arena_bytes(cfg: sekv_config):
    dev, slot = C.c_size_t(0), C.c_size_t(0)
    st = lib.sekv_device_arena_bytes(C.byref(cfg), C.byref(dev), C.byref(slot))
    if st != SEKV_OK:
        raise SekvError(st, "sekv_device_arena_bytes")
    return int(dev.value), int(slot.value)


def sekv_build_sizes(cfg: sekv_config, seq_tok_off: Sequence[int], H: Optional[torch.Tensor] = None):
    """(sekv_sizes, spans_per_seq, pool_per_seq) for a batch before any handle exists: exact when the DEVICE
    surprisal tensor H is given (the segmentation rule runs on the GPU), upper bounds from token counts otherwise."""
    n = len(seq_tok_off) - 1
    off = (C.c_int64 * (n + 1))(*[int(x) for x in seq_tok_off])
    out = sekv_sizes()
    spans, pool = (C.c_int32 * n)(), (C.c_int32 * n)()
    if H is not None:
        assert H.is_cuda and H.dtype == torch.float32 and H.is_contiguous()
        torch.cuda.synchronize(H.device)
    st = lib.sekv_build_sizes(C.byref(cfg), n, off, None if H is None else H.data_ptr(), C.byref(out), spans, pool)
    if st != SEKV_OK:
        raise SekvError(st, "sekv_build_sizes")
    return out, list(spans), list(pool)


SEKV_STATIC_MAX_TOKENS = 1 << 20
SEKV_STATIC_MAX_SEQS = 1024


def sekv_segment_counts_static(cfg: sekv_config, seq_tok_off: Sequence[int], H: torch.Tensor, counts: torch.Tensor,
                               too_long: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> None:
    """Per-sequence (pool tokens, spans) into the DEVICE int32 tensor counts [n_seqs, 2] and the span-too-long flag into
    the DEVICE int32 tensor too_long [1], on scratch the library holds in a static device array: nothing is allocated
    (include/sekv.h).  Asynchronous on `stream` (default: torch's current stream)."""
    n = len(seq_tok_off) - 1
    off = (C.c_int64 * (n + 1))(*[int(x) for x in seq_tok_off])
    assert H.is_cuda and H.dtype == torch.float32 and H.is_contiguous()
    assert counts.is_cuda and counts.dtype == torch.int32 and counts.is_contiguous() and counts.numel() >= 2 * n
    assert too_long.is_cuda and too_long.dtype == torch.int32 and too_long.numel() >= 1
    s = stream if stream is not None else torch.cuda.current_stream(H.device)
    with torch.cuda.device(H.device):
        st = lib.sekv_segment_counts_static(C.byref(cfg), n, off, H.data_ptr(), counts.data_ptr(), too_long.data_ptr(),
                                            s.cuda_stream)
    if st != SEKV_OK:
        raise SekvError(st, "sekv_segment_counts_static: " + lib.sekv_static_last_error().decode())


def make_config(**kw) -> sekv_config:
    """Config with the paper's defaults: alpha 1.0, l_min 16, d' 32, R_max 32."""
    d = dict(n_layers=1, n_q_heads=32, n_kv_heads=8, head_dim=128, route_dim=32, dtype=SEKV_BF16,
             out_dtype=SEKV_F32, alpha=1.0, l_min=16, r_max=32, window=0, max_seqs=1, max_tokens_total=1,
             max_spans_total=1, max_full_total=1, max_span_len=256, k_cap=16, cache_ways=32, prefetch=0, stage1_ctas=0,
             item_rows=0, zoom_spans_per_item=0, use_graph=0, impl=0, main_stream=None, side_stream=None)
    unknown = set(kw) - set(d)
    if unknown:
        raise TypeError(f"unknown config fields {sorted(unknown)}")
    d.update(kw)
    return sekv_config(**d)


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    if t is None:
        return None
    assert t.is_contiguous(), "tensors crossing the C ABI must be contiguous"
    return t.data_ptr()


_MAIN_STREAMS: dict = {}


def main_stream(device: torch.device) -> "torch.cuda.Stream":
    """One non-default stream per device, made torch's current stream: the library launches on it (and
    can capture CUDA graphs on it, which the legacy default stream does not allow), and torch ops
    issued by the caller are ordered with the library's kernels because they share the stream."""
    key = torch.device(device).index or 0
    if key not in _MAIN_STREAMS:
        _MAIN_STREAMS[key] = torch.cuda.Stream(device)
    torch.cuda.set_stream(_MAIN_STREAMS[key])
    return _MAIN_STREAMS[key]


class Sekv:
    """Owner of one sekv_handle plus the two arenas it borrows.  Method names follow the C calls."""

    def __init__(self, cfg: sekv_config, host_bytes: int, device: str = "cuda:0"):
        self.cfg = cfg
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        torch.cuda.synchronize(self.device)
        self._main = main_stream(self.device)
        self._side = torch.cuda.Stream(self.device)
        cfg.main_stream = self._main.cuda_stream
        cfg.side_stream = self._side.cuda_stream
        dev_bytes, self.slot_bytes = sekv_device_arena_bytes(cfg)
        self.dev_arena = torch.empty(dev_bytes + 256, dtype=torch.uint8, device=self.device)
        off = (-self.dev_arena.data_ptr()) % 256
        self.dev_arena = self.dev_arena[off:off + dev_bytes]
        # Page-aligned pageable host memory; sekv_create page-locks and device-maps it
        # (cudaHostRegister) -- torch's pin_memory would round 16 GB up to 32 GB.
        host_bytes = max(int(host_bytes), 4096)
        self._host_raw = torch.empty(host_bytes + 4096, dtype=torch.uint8)
        hoff = (-self._host_raw.data_ptr()) % 4096
        self.host_arena = self._host_raw[hoff:hoff + host_bytes]
        h = C.c_void_p(None)
        st = lib.sekv_create(C.byref(cfg), self.dev_arena.data_ptr(), dev_bytes, self.host_arena.data_ptr(),
                             host_bytes, C.byref(h))
        if st != SEKV_OK:
            raise SekvError(st, "sekv_create")
        self._h = h
        self.esize = 2 if cfg.dtype == SEKV_BF16 else 4
        self.st_dtype = torch.bfloat16 if cfg.dtype == SEKV_BF16 else torch.float32
        self.out_dtype = torch.bfloat16 if cfg.out_dtype == SEKV_BF16 else torch.float32
        self.n_seqs = 0
        self.spans_per_seq: list = []
        self.pool_per_seq: list = []

    # -- helpers ---------------------------------------------------------------------------------
    def _check(self, st: int, where: str):
        if st != SEKV_OK:
            raise SekvError(st, where, lib.sekv_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            lib.sekv_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- a0 -----------------------------------------------------------------------------------------
    def _seq_off(self, seq_tok_off: Sequence[int]):
        n = len(seq_tok_off) - 1
        return n, (C.c_int64 * (n + 1))(*[int(x) for x in seq_tok_off])

    def _after_build(self, n, spans, pool):
        self.n_seqs = n
        self.spans_per_seq = list(spans)
        self.pool_per_seq = list(pool)

    def sekv_build_spans(self, layer: int, seq_tok_off: Sequence[int], H: torch.Tensor, K: torch.Tensor,
                         V: torch.Tensor, W: torch.Tensor, rank_cap: int = 0):
        n, off = self._seq_off(seq_tok_off)
        spans, pool = (C.c_int32 * n)(), (C.c_int32 * n)()
        st = lib.sekv_build_spans(self._h, layer, n, off, _ptr(H), _ptr(K), _ptr(V), _ptr(W), rank_cap, spans, pool)
        self._check(st, "sekv_build_spans")
        self._after_build(n, spans, pool)

    def sekv_build_spans_prefactored(self, layer: int, seq_tok_off: Sequence[int], H: torch.Tensor, *, rank_in: int,
                                     tokUK, SK, VtK, tokUV, SV, VtV, Kfull, Vfull, W, rank_k=None, rank_v=None,
                                     a_tot: int, m_tot: int):
        n, off = self._seq_off(seq_tok_off)
        f = sekv_factors(rank_in=rank_in, tokUK=_ptr(tokUK), SK=_ptr(SK), VtK=_ptr(VtK), tokUV=_ptr(tokUV),
                         SV=_ptr(SV), VtV=_ptr(VtV), rank_k=_ptr(rank_k), rank_v=_ptr(rank_v), Kfull=_ptr(Kfull),
                         Vfull=_ptr(Vfull), a_tot=a_tot, m_tot=m_tot)
        spans, pool = (C.c_int32 * n)(), (C.c_int32 * n)()
        st = lib.sekv_build_spans_prefactored(self._h, layer, n, off, _ptr(H), C.byref(f), _ptr(W), spans, pool)
        self._check(st, "sekv_build_spans_prefactored")
        self._after_build(n, spans, pool)

    def sekv_reset(self):
        self._check(lib.sekv_reset(self._h), "sekv_reset")
        self.n_seqs = 0

    # -- a1-a3 ------------------------------------------------------------------------------------------
    def sekv_route(self, layer: int, q: torch.Tensor, k: int, tau: Optional[torch.Tensor] = None,
                   logits: Optional[torch.Tensor] = None, alpha_tilde: Optional[torch.Tensor] = None,
                   ids: Optional[torch.Tensor] = None, count: Optional[torch.Tensor] = None):
        kc = max(self.cfg.k_cap, 1)
        if ids is None:
            ids = torch.empty((self.n_seqs, self.cfg.n_kv_heads, kc), dtype=torch.int32, device=self.device)
        if count is None:
            count = torch.empty((self.n_seqs, self.cfg.n_kv_heads), dtype=torch.int32, device=self.device)
        st = lib.sekv_route(self._h, layer, _ptr(q), _ptr(tau), k, _ptr(logits), _ptr(alpha_tilde), _ptr(ids), _ptr(count))
        self._check(st, "sekv_route")
        return ids, count

    # -- a4-a7 --------------------------------------------------------------------------------------------
    def sekv_decode_attn(self, layer: int, q: torch.Tensor, ids: Optional[torch.Tensor], count: Optional[torch.Tensor],
                         out: Optional[torch.Tensor] = None, lse: Optional[torch.Tensor] = None):
        if out is None:
            out = torch.empty((self.n_seqs, self.cfg.n_q_heads, 128), dtype=self.out_dtype, device=self.device)
        st = lib.sekv_decode_attn(self._h, layer, _ptr(q), _ptr(ids), _ptr(count), _ptr(out), _ptr(lse))
        self._check(st, "sekv_decode_attn")
        return out

    def sekv_decode_step(self, q: torch.Tensor, k: int, out: torch.Tensor, tau: Optional[torch.Tensor] = None,
                         lse: Optional[torch.Tensor] = None):
        st = lib.sekv_decode_step(self._h, _ptr(q), _ptr(tau), k, _ptr(out), _ptr(lse))
        self._check(st, "sekv_decode_step")
        return out

    def sekv_last_zoom_ids(self, layer: int):
        kc = max(self.cfg.k_cap, 1)
        ids = torch.empty((self.n_seqs, self.cfg.n_kv_heads, kc), dtype=torch.int32, device=self.device)
        count = torch.empty((self.n_seqs, self.cfg.n_kv_heads), dtype=torch.int32, device=self.device)
        self._check(lib.sekv_last_zoom_ids(self._h, layer, _ptr(ids), _ptr(count)), "sekv_last_zoom_ids")
        return ids, count

    def sekv_decode_step_host(self, q_host: torch.Tensor, k: int, out_host: torch.Tensor,
                              tau: Optional[torch.Tensor] = None, lse_host: Optional[torch.Tensor] = None):
        assert not q_host.is_cuda and not out_host.is_cuda
        st = lib.sekv_decode_step_host(self._h, _ptr(q_host), _ptr(tau), k, _ptr(out_host), _ptr(lse_host))
        self._check(st, "sekv_decode_step_host")
        return out_host

    # -- introspection ---------------------------------------------------------------------------------------
    def sekv_get_layout(self) -> sekv_layout:
        lay = sekv_layout()
        self._check(lib.sekv_get_layout(self._h, C.byref(lay)), "sekv_get_layout")
        return lay

    def sekv_get_stats(self) -> dict:
        s = sekv_stats()
        self._check(lib.sekv_get_stats(self._h, C.byref(s)), "sekv_get_stats")
        return {n: int(getattr(s, n)) for n in _STATS_FIELDS}

    def sekv_reset_stats(self):
        self._check(lib.sekv_reset_stats(self._h), "sekv_reset_stats")

    def sekv_cache_flush(self):
        self._check(lib.sekv_cache_flush(self._h), "sekv_cache_flush")

    def sekv_static_bytes_per_layer(self) -> int:
        v = C.c_uint64(0)
        self._check(lib.sekv_static_bytes_per_layer(self._h, C.byref(v)), "sekv_static_bytes_per_layer")
        return int(v.value)

    KERNEL_CLASSES = ("route", "plan", "fetch", "stage1", "stage2", "combine", "fused", "prefetch")

    def sekv_set_profiling(self, on: bool):
        self._check(lib.sekv_set_profiling(self._h, 1 if on else 0), "sekv_set_profiling")

    def sekv_get_kernel_times(self) -> dict:
        ms, n = (C.c_double * 8)(), (C.c_uint64 * 8)()
        self._check(lib.sekv_get_kernel_times(self._h, ms, n), "sekv_get_kernel_times")
        return {name: dict(ms=float(ms[i]), launches=int(n[i])) for i, name in enumerate(self.KERNEL_CLASSES)}

    def sekv_set_trace(self, buf: Optional[torch.Tensor]) -> int:
        """buf: uint8/int64 DEVICE tensor of 64 bytes per item, or None to switch tracing off."""
        n = C.c_int32(0)
        cap = 0 if buf is None else buf.numel() * buf.element_size() // 64
        self._check(lib.sekv_set_trace(self._h, _ptr(buf), cap, C.byref(n)), "sekv_set_trace")
        self._trace_buf = buf
        return int(n.value)

    def sekv_graph_count(self) -> int:
        n = C.c_int32(0)
        self._check(lib.sekv_graph_count(self._h, C.byref(n)), "sekv_graph_count")
        return int(n.value)

    def sekv_get_path(self):
        """(fused, reason): whether the built batch runs on the fused layer kernel, and why not if it does not."""
        f, why = C.c_int32(0), C.c_char_p(None)
        self._check(lib.sekv_get_path(self._h, C.byref(f), C.byref(why)), "sekv_get_path")
        return bool(f.value), (why.value or b"").decode()

    def sekv_export_span_factors(self, layer: int, seq: int, kv_head: int, span: int) -> dict:
        """One span's factors decoded by the library into row-major float32 numpy arrays."""
        import numpy as np
        ln, rk, rv, pad = C.c_int32(0), C.c_int32(0), C.c_int32(0), C.c_int32(0)
        st = lib.sekv_export_span_factors(self._h, layer, seq, kv_head, span, C.byref(ln), C.byref(rk), C.byref(rv),
                                          None, None, None, None, None, None, None)
        self._check(st, "sekv_export_span_factors")
        n, a, b = ln.value, rk.value, rv.value
        arr = dict(UK=np.zeros((n, a), np.float32), sK=np.zeros(a, np.float32), VtK=np.zeros((a, 128), np.float32),
                   UV=np.zeros((n, b), np.float32), sV=np.zeros(b, np.float32), VtV=np.zeros((b, 128), np.float32))
        ptr = lambda x: x.ctypes.data_as(C.c_void_p)
        st = lib.sekv_export_span_factors(self._h, layer, seq, kv_head, span, C.byref(ln), C.byref(rk), C.byref(rv),
                                          ptr(arr["UK"]), ptr(arr["sK"]), ptr(arr["VtK"]), ptr(arr["UV"]),
                                          ptr(arr["sV"]), ptr(arr["VtV"]), C.byref(pad))
        self._check(st, "sekv_export_span_factors")
        arr["pad_ok"] = bool(pad.value)
        return arr

    def sekv_get_schedule(self):
        a, b = C.c_int32(0), C.c_int32(0)
        self._check(lib.sekv_get_schedule(self._h, C.byref(a), C.byref(b)), "sekv_get_schedule")
        return int(a.value), int(b.value)
