// C-ABI entry points of libsekv: handle, arena layout, build / route / decode orchestration.
// Every step of the path runs in the CUDA kernels of the other translation units; this file holds
// argument checking, memory layout, stream/event/graph plumbing and allocation bookkeeping only.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "sekv_internal.cuh"

using namespace sekv;

namespace {

constexpr size_t kAlign = 256;

struct Carver {
  size_t off = 0;
  int64_t take(size_t bytes) {
    off = round_up_sz(off, kAlign);
    int64_t o = (int64_t)off;
    off += bytes;
    return o;
  }
};

const char* check_config(const sekv_config* c) {
  if (!c) return "config is NULL";
  if (c->n_layers < 1) return "n_layers < 1";
  if (c->head_dim != SEKV_HEAD_DIM) return "head_dim must be 128";
  if (c->n_kv_heads < 1 || c->n_q_heads < 1 || c->n_q_heads % c->n_kv_heads) return "n_q_heads must be a multiple of n_kv_heads";
  if (c->n_q_heads / c->n_kv_heads > SEKV_MAX_GROUP) return "more than 8 query heads per kv head";
  if (c->route_dim < 8 || c->route_dim > SEKV_MAX_ROUTE_DIM || c->route_dim % 8) return "route_dim must be a multiple of 8 in [8, 64]";
  if (c->dtype != SEKV_F32 && c->dtype != SEKV_BF16) return "dtype must be SEKV_F32 or SEKV_BF16";
  if (c->out_dtype != SEKV_F32 && c->out_dtype != SEKV_BF16) return "out_dtype must be SEKV_F32 or SEKV_BF16";
  if (c->l_min < 1) return "l_min < 1";
  if (c->r_max < 1 || c->r_max > SEKV_MAX_RANK) return "r_max must be in [1, 64]";
  if (c->window < 0) return "window < 0";
  if (c->max_seqs < 1) return "max_seqs < 1";
  if (c->max_tokens_total < 1) return "max_tokens_total < 1";
  if (c->max_spans_total < 1 || c->max_full_total < 0) return "bad span / pool capacity";
  if (c->max_span_len < 1 || c->max_span_len > SEKV_MAX_SPAN_LEN) return "max_span_len must be in [1, 1024]";
  if (c->k_cap < 0) return "k_cap < 0";
  if (c->prefetch < 0 || c->prefetch > 1024) return "prefetch must be in [0, 1024]";
  if (c->cache_ways < std::max(c->k_cap, 1) + c->prefetch) return "cache_ways must be >= max(k_cap, 1) + prefetch";
  if (c->item_rows < 0 || c->item_rows % 16) return "item_rows must be a non-negative multiple of 16";
  if (c->zoom_spans_per_item < 0 || c->zoom_spans_per_item > 64) return "zoom_spans_per_item must be in [0, 64]";
  if (c->cache_ways > 8192) return "cache_ways > 8192";
  if (c->stage1_ctas < 0 || c->stage1_ctas > 4096) return "stage1_ctas out of range";
  if (!(c->alpha == c->alpha)) return "alpha is NaN";
  return nullptr;
}

void compute_layout(const sekv_config& c, FullLayout* F) {
  memset(F, 0, sizeof(*F));
  sekv_layout& L = F->lay;
  const int64_t es = c.dtype == SEKV_BF16 ? 2 : 4;
  const int64_t B = c.max_seqs, Hq = c.n_q_heads, Hkv = c.n_kv_heads, NL = c.n_layers;
  const int64_t mcap = c.max_spans_total, acap = c.max_full_total, rcap = mcap + acap;
  const int kcap = std::max(c.k_cap, 1);
  const int kc = kcap + std::max(c.prefetch, 0);
  L.esize = es; L.rows_cap = rcap; L.spans_cap = mcap;
  Carver cv;
  L.seq_tok_off = cv.take((B + 1) * 8);
  L.seq_row_off = cv.take((B + 1) * 4);
  L.seq_span_off = cv.take((B + 1) * 4);
  L.seq_pool_cnt = cv.take(B * 4);
  L.span_len = cv.take(mcap * 4);
  L.span_tok_start = cv.take(mcap * 8);
  L.ln_len = cv.take(mcap * 4);
  L.pool_tok = cv.take(std::max<int64_t>(acap, 1) * 8);
  L.ent_head_stride = rcap * kD * es;
  L.ent_layer_stride = round_up_sz(Hkv * L.ent_head_stride, kAlign);
  L.ent_k = cv.take(NL * L.ent_layer_stride);
  L.ent_v = cv.take(NL * L.ent_layer_stride);
  L.route_head_stride = mcap * c.route_dim * es;
  L.route_layer_stride = round_up_sz(Hq * L.route_head_stride, kAlign);
  L.route = cv.take(NL * L.route_layer_stride);
  L.w_layer_stride = round_up_sz(Hq * c.route_dim * kD * es, kAlign);
  L.w = cv.take(NL * L.w_layer_stride);
  L.dir_layer_stride_elems = Hkv * mcap;
  L.dir_off = cv.take(NL * L.dir_layer_stride_elems * 8);
  L.dir_rank = cv.take(NL * L.dir_layer_stride_elems * 4);
  const int64_t regions = NL * B * Hkv;
  L.cache_tags = cv.take(regions * c.cache_ways * 4);
  L.cache_stamps = cv.take(regions * c.cache_ways * 4);
  BlobDims bd = blob_dims((int)es, c.max_span_len, c.r_max, c.r_max);
  L.slot_bytes = (int64_t)bd.bytes;
  L.cache_slots = cv.take((size_t)regions * c.cache_ways * bd.bytes);
  // workspace
  // capacity of the stage-1 chunk list (generic path) and of the fused kernel's item list (row items of
  // >= 16 rows, one expanded span per ZOOM item at the finest)
  const int64_t attn_items = Hkv * (rcap / 16 + 2 * B + 2) + B * Hkv * kcap;
  F->max_chunks = (int)std::max<int64_t>(std::max(c.stage1_ctas, 1024) + B * Hkv, attn_items);
  F->max_items = (int)(attn_items + 2 * B * Hq + B * Hkv * (1 + std::max(c.prefetch, 0)) + Hkv * (mcap / 8 + B + 1));
  const int G = c.n_q_heads / c.n_kv_heads;
  const int P2 = (kcap + kStage2SpansPerCta - 1) / kStage2SpansPerCta;
  F->off_partials1 = cv.take((size_t)F->max_chunks * G * kPartStride * 4);
  F->off_partials2 = cv.take((size_t)B * Hkv * P2 * G * kPartStride * 4);
  F->off_ws_ids = cv.take((size_t)NL * B * Hkv * kcap * 4);
  F->off_ws_count = cv.take((size_t)NL * B * Hkv * 4);
  F->off_stats = cv.take(ST_COUNT * 8);
  F->off_chunks = cv.take((size_t)F->max_chunks * sizeof(Chunk));
  F->off_bg_chunk = cv.take((size_t)(B * Hkv + 1) * 4);
  F->mask_words = (int)((std::min<int64_t>(mcap, SEKV_MAX_SPANS_PER_SEQ) + 31) / 32);
  F->off_zoom_mask = cv.take((size_t)NL * B * Hkv * F->mask_words * 4);
  F->off_items = cv.take((size_t)NL * B * Hkv * kc * 4);
  F->off_item_span = cv.take((size_t)NL * B * Hkv * kc * 4);
  F->off_items_sched = cv.take((size_t)F->max_items * sizeof(Item));
  F->off_bg_part = cv.take((size_t)(B * Hkv + 1) * 8);          // int2 per group: first span, span count
  F->off_bg_route = cv.take((size_t)(B * Hkv) * 4);
  F->ctrs_per_layer = (int)(4 + 2 * (4 + 4 * B * Hkv));       // sequence number + two counter sets
  F->off_zdesc = cv.take((size_t)NL * B * Hkv * kc * sizeof(ZDescG));
  F->off_zway = cv.take((size_t)NL * B * Hkv * kc * sizeof(uint2));
  F->off_zmask2 = cv.take((size_t)NL * B * Hkv * F->mask_words * 8);
  F->off_ctrs = cv.take((size_t)NL * F->ctrs_per_layer * 4);
  F->off_plan_counts = cv.take((size_t)NL * B * Hkv * 2 * 4);
  F->off_layer_step = cv.take((size_t)NL * 4);
  F->off_seg_flag = cv.take((size_t)c.max_tokens_total);
  F->off_seg_flag2 = cv.take((size_t)c.max_tokens_total);
  F->off_seg_len = cv.take((size_t)c.max_tokens_total * 4);
  F->off_seg_misc = cv.take((size_t)B * 32);
  F->off_err_flag = cv.take(16);
  const int64_t osz = c.out_dtype == SEKV_BF16 ? 2 : 4;
  F->off_q_stage = cv.take((size_t)NL * B * Hq * kD * es);
  F->off_out_stage = cv.take((size_t)NL * B * Hq * kD * osz);
  F->off_lse_stage = cv.take((size_t)NL * B * Hq * 4);
  F->total = round_up_sz(cv.off, kAlign);
  L.device_bytes_total = (int64_t)F->total;
}

sekv_status fail(sekv_handle* h, sekv_status s, const std::string& msg) {
  if (h) h->err = msg;
  return s;
}
sekv_status cuda_fail(sekv_handle* h, cudaError_t e, const char* where) {
  char buf[256];
  snprintf(buf, sizeof(buf), "%s: %s", where, cudaGetErrorString(e));
  return fail(h, SEKV_CUDA, buf);
}
#define CK(h, expr)                                          \
  do {                                                       \
    cudaError_t e__ = (expr);                                \
    if (e__ != cudaSuccess) return cuda_fail(h, e__, #expr); \
  } while (0)

}  // namespace

namespace sekv {

CsrView csr_view(const sekv_handle* h) {
  CsrView v;
  uint8_t* d = h->dev;
  v.seq_tok_off = (const int64_t*)(d + h->lay.seq_tok_off);
  v.seq_row_off = (const int32_t*)(d + h->lay.seq_row_off);
  v.seq_span_off = (const int32_t*)(d + h->lay.seq_span_off);
  v.seq_pool_cnt = (const int32_t*)(d + h->lay.seq_pool_cnt);
  v.span_len = (const int32_t*)(d + h->lay.span_len);
  v.span_tok_start = (const int64_t*)(d + h->lay.span_tok_start);
  v.ln_len = (const float*)(d + h->lay.ln_len);
  v.pool_tok = (const int64_t*)(d + h->lay.pool_tok);
  return v;
}

LayerView layer_view(const sekv_handle* h, int l) {
  LayerView v;
  uint8_t* d = h->dev;
  const sekv_layout& L = h->lay;
  const sekv_config& c = h->cfg;
  const int64_t B = c.max_seqs, Hkv = c.n_kv_heads;
  const int kcap = std::max(c.k_cap, 1) + std::max(c.prefetch, 0);
  v.ent_k = d + L.ent_k + (int64_t)l * L.ent_layer_stride;
  v.ent_v = d + L.ent_v + (int64_t)l * L.ent_layer_stride;
  v.route = d + L.route + (int64_t)l * L.route_layer_stride;
  v.W = d + L.w + (int64_t)l * L.w_layer_stride;
  v.dir_off = (const int64_t*)(d + L.dir_off) + (int64_t)l * L.dir_layer_stride_elems;
  v.dir_rank = (const int32_t*)(d + L.dir_rank) + (int64_t)l * L.dir_layer_stride_elems;
  const int64_t region0 = (int64_t)l * B * Hkv;
  v.tags = (int32_t*)(d + L.cache_tags) + region0 * c.cache_ways;
  v.stamps = (uint32_t*)(d + L.cache_stamps) + region0 * c.cache_ways;
  v.slots = d + L.cache_slots + (size_t)region0 * c.cache_ways * L.slot_bytes;
  v.layer_step = (uint32_t*)(d + h->F.off_layer_step) + l;
  v.zoom_mask = (uint32_t*)(d + h->F.off_zoom_mask) + region0 * h->mask_words;
  v.items = (uint32_t*)(d + h->F.off_items) + region0 * kcap;
  v.item_span = (int32_t*)(d + h->F.off_item_span) + region0 * kcap;
  return v;
}

}  // namespace sekv

extern "C" {

const char* sekv_version(void) { return "sekv-b200 0.1 (sm_100a)"; }

const char* sekv_status_string(sekv_status s) {
  switch (s) {
    case SEKV_OK: return "SEKV_OK";
    case SEKV_INVALID_ARG: return "SEKV_INVALID_ARG";
    case SEKV_UNSUPPORTED: return "SEKV_UNSUPPORTED";
    case SEKV_OOM_DEVICE: return "SEKV_OOM_DEVICE";
    case SEKV_OOM_HOST: return "SEKV_OOM_HOST";
    case SEKV_CUDA: return "SEKV_CUDA";
    case SEKV_STATE: return "SEKV_STATE";
  }
  return "SEKV_?";
}

sekv_status sekv_device_arena_bytes(const sekv_config* cfg, size_t* device_bytes, size_t* slot_bytes) {
  if (check_config(cfg)) return SEKV_INVALID_ARG;
  FullLayout F;
  compute_layout(*cfg, &F);
  if (device_bytes) *device_bytes = F.total;
  if (slot_bytes) *slot_bytes = (size_t)F.lay.slot_bytes;
  return SEKV_OK;
}

size_t sekv_blob_bytes(int32_t dtype, int32_t span_len, int32_t rank_k, int32_t rank_v) {
  return blob_dims(dtype == SEKV_BF16 ? 2 : 4, span_len, rank_k, rank_v).bytes;
}

sekv_status sekv_build_sizes(const sekv_config* cfg, int32_t n_seqs, const int64_t* seq_tok_off, const float* H,
                             sekv_sizes* out, int32_t* spans_per_seq, int32_t* pool_per_seq) {
  if (!cfg || !out || !seq_tok_off || n_seqs < 1) return SEKV_INVALID_ARG;
  if (cfg->l_min < 1 || cfg->r_max < 1 || cfg->r_max > SEKV_MAX_RANK || cfg->n_layers < 1 || cfg->n_kv_heads < 1 ||
      cfg->window < 0 || !(cfg->alpha == cfg->alpha))
    return SEKV_INVALID_ARG;
  if (seq_tok_off[0] != 0) return SEKV_INVALID_ARG;
  for (int b = 0; b < n_seqs; ++b)
    if (seq_tok_off[b + 1] <= seq_tok_off[b]) return SEKV_INVALID_ARG;
  memset(out, 0, sizeof(*out));
  const int es = cfg->dtype == SEKV_BF16 ? 2 : 4;
  const int64_t n_tot = seq_tok_off[n_seqs];
  const int64_t per_store = (int64_t)cfg->n_layers * cfg->n_kv_heads;
  out->tokens_total = n_tot;
  if (!H) {
    int64_t m = 0, longest = 0, bytes = 0;
    for (int b = 0; b < n_seqs; ++b) {
      const int64_t n = seq_tok_off[b + 1] - seq_tok_off[b];
      const int64_t mb = n / cfg->l_min;
      m += mb; longest = std::max(longest, n);
      out->max_spans_per_seq = (int32_t)std::max<int64_t>(out->max_spans_per_seq, mb);
      if (spans_per_seq) spans_per_seq[b] = (int32_t)mb;
      if (pool_per_seq) pool_per_seq[b] = (int32_t)n;
      // the most expensive cover of n tokens: spans of exactly l_min tokens (largest header share)
      bytes += mb * (int64_t)blob_dims(es, cfg->l_min, std::min(cfg->r_max, cfg->l_min), std::min(cfg->r_max, cfg->l_min)).bytes
               + (int64_t)blob_dims(es, (int)std::min<int64_t>(n, SEKV_MAX_SPAN_LEN), 1, 1).chunk_bytes;
    }
    if (m > INT32_MAX || n_tot > INT32_MAX) return SEKV_UNSUPPORTED;
    out->spans_total = (int32_t)m; out->full_total = (int32_t)n_tot;
    out->max_span_len = (int32_t)std::min<int64_t>(longest, SEKV_MAX_SPAN_LEN);
    out->exact = 0;
    out->host_bytes = bytes * per_store + (1 << 16);
    return SEKV_OK;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return SEKV_CUDA; }
  // scratch: flags (2 bytes per token), run lengths (4), token offsets, thresholds, counts, error flag
  const size_t o_flag2 = round_up_sz((size_t)n_tot, 256), o_len = o_flag2 + round_up_sz((size_t)n_tot, 256);
  const size_t o_off = o_len + round_up_sz((size_t)n_tot * 4, 256), o_thr = o_off + round_up_sz((size_t)(n_seqs + 1) * 8, 256);
  const size_t o_cnt = o_thr + round_up_sz((size_t)n_seqs * 8, 256), o_err = o_cnt + round_up_sz((size_t)n_seqs * 8, 256);
  uint8_t* tmp = nullptr;
  if (cudaMalloc(&tmp, o_err + 256) != cudaSuccess) { cudaGetLastError(); return SEKV_OOM_DEVICE; }
  sekv_status st = SEKV_OK;
  std::vector<int32_t> cnt((size_t)n_seqs * 2);
  std::vector<uint8_t> f2((size_t)n_tot);
  std::vector<int32_t> len_at((size_t)n_tot);
  int herr = 0;
  cudaError_t e = cudaMemcpy(tmp + o_off, seq_tok_off, (size_t)(n_seqs + 1) * 8, cudaMemcpyHostToDevice);
  if (e == cudaSuccess)
    e = segment_scan(H, n_seqs, (const int64_t*)(tmp + o_off), (double)cfg->alpha, cfg->window, cfg->l_min, SEKV_MAX_SPAN_LEN,
                     tmp, tmp + o_flag2, (int32_t*)(tmp + o_len), (double*)(tmp + o_thr), (int32_t*)(tmp + o_cnt),
                     (int*)(tmp + o_err), 0);
  if (e == cudaSuccess) e = cudaMemcpy(cnt.data(), tmp + o_cnt, cnt.size() * 4, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(&herr, tmp + o_err, 4, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(f2.data(), tmp + o_flag2, (size_t)n_tot, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(len_at.data(), tmp + o_len, (size_t)n_tot * 4, cudaMemcpyDeviceToHost);
  cudaFree(tmp);
  if (e != cudaSuccess) { cudaGetLastError(); return SEKV_CUDA; }
  if (herr) return SEKV_UNSUPPORTED;                          // a run longer than SEKV_MAX_SPAN_LEN
  int64_t m = 0, a = 0, bytes = 0;
  int longest = 1;
  for (int b = 0; b < n_seqs; ++b) {
    a += cnt[b * 2]; m += cnt[b * 2 + 1];
    out->max_spans_per_seq = std::max(out->max_spans_per_seq, cnt[b * 2 + 1]);
    if (spans_per_seq) spans_per_seq[b] = cnt[b * 2 + 1];
    if (pool_per_seq) pool_per_seq[b] = cnt[b * 2];
  }
  for (int64_t t = 0; t < n_tot; ++t)
    if (f2[t] == 3) {                                          // first token of a span: its length is recorded there
      const int len = len_at[t], r = std::min(cfg->r_max, len);
      longest = std::max(longest, len);
      bytes += (int64_t)blob_dims(es, len, r, r).bytes;
    }
  out->spans_total = (int32_t)m; out->full_total = (int32_t)a; out->max_span_len = longest; out->exact = 1;
  out->host_bytes = bytes * per_store + (1 << 16);
  return st;
}

sekv_status sekv_create(const sekv_config* cfg, void* device_arena, size_t device_bytes, void* host_arena,
                        size_t host_bytes, sekv_handle** out) {
  if (!out) return SEKV_INVALID_ARG;
  *out = nullptr;
  if (check_config(cfg)) return SEKV_INVALID_ARG;
  if (!device_arena || ((uintptr_t)device_arena % kAlign)) return SEKV_INVALID_ARG;
  if (!host_arena || ((uintptr_t)host_arena % 128)) return SEKV_INVALID_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return SEKV_CUDA; }
  sekv_handle* h = new (std::nothrow) sekv_handle();
  if (!h) return SEKV_OOM_HOST;
  h->registered_host = false;
  h->cfg = *cfg;
  h->G = cfg->n_q_heads / cfg->n_kv_heads;
  h->esize = cfg->dtype == SEKV_BF16 ? 2 : 4;
  compute_layout(*cfg, &h->F);
  h->lay = h->F.lay;
  if (device_bytes < h->F.total) { delete h; return SEKV_OOM_DEVICE; }
  h->dev = (uint8_t*)device_arena; h->dev_bytes = device_bytes;
  h->host = (uint8_t*)host_arena; h->host_bytes = host_bytes;
  const FullLayout& F = h->F;
  h->mask_words = F.mask_words;
  h->main = (cudaStream_t)cfg->main_stream;
  h->side = (cudaStream_t)cfg->side_stream;
  h->own_side = false;
  cudaError_t e;
  void* hd = nullptr;
  e = cudaHostGetDevicePointer(&hd, host_arena, 0);
  if (e != cudaSuccess) {
    cudaGetLastError();
    e = cudaHostRegister(host_arena, host_bytes, cudaHostRegisterMapped | cudaHostRegisterPortable);
    if (e == cudaSuccess) { h->registered_host = true; e = cudaHostGetDevicePointer(&hd, host_arena, 0); }
  }
  if (e != cudaSuccess) { cudaGetLastError(); if (h->registered_host) cudaHostUnregister(host_arena); delete h; return SEKV_CUDA; }
  h->host_dev = (uint8_t*)hd;
  if (!h->side) {
    if (cudaStreamCreateWithFlags(&h->side, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); delete h; return SEKV_CUDA; }
    h->own_side = true;
  }
  cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming);
  cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming);
  int dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev);
  h->launches = 0;
  h->profiling = false;
  h->trace_buf = nullptr; h->trace_cap = 0;
  h->use_pdl = true;
  *out = h;
  sekv_status s = sekv_reset(h);
  if (s != SEKV_OK) { sekv_destroy(h); *out = nullptr; return s; }
  return SEKV_OK;
}

void sekv_destroy(sekv_handle* h) {
  if (!h) return;
  cudaStreamSynchronize(h->main);
  cudaStreamSynchronize(h->side);
  for (auto& g : h->graphs) cudaGraphExecDestroy(g.exec);
  for (auto& r : h->prof) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
  if (h->own_side) cudaStreamDestroy(h->side);
  cudaEventDestroy(h->ev_fork);
  cudaEventDestroy(h->ev_join);
  if (h->registered_host) cudaHostUnregister(h->host);
  delete h;
}

const char* sekv_last_error(const sekv_handle* h) { return h ? h->err.c_str() : "null handle"; }

sekv_status sekv_reset(sekv_handle* h) {
  if (!h) return SEKV_INVALID_ARG;
  const FullLayout& F = h->F;
  const sekv_config& c = h->cfg;
  CK(h, cudaStreamSynchronize(h->main));
  CK(h, cudaStreamSynchronize(h->side));
  for (auto& g : h->graphs) cudaGraphExecDestroy(g.exec);
  h->graphs.clear();
  const int64_t regions = (int64_t)c.n_layers * c.max_seqs * c.n_kv_heads;
  CK(h, cudaMemsetAsync(h->dev + h->lay.cache_tags, 0xFF, regions * c.cache_ways * 4, h->main));
  CK(h, cudaMemsetAsync(h->dev + h->lay.cache_stamps, 0, regions * c.cache_ways * 4, h->main));
  CK(h, cudaMemsetAsync(h->dev + F.off_layer_step, 0, (size_t)c.n_layers * 4, h->main));
  CK(h, cudaMemsetAsync(h->dev + F.off_zdesc, 0, (size_t)c.n_layers * c.max_seqs * c.n_kv_heads *
                        (std::max(c.k_cap, 1) + std::max(c.prefetch, 0)) * sizeof(ZDescG), h->main));   // stamps restart
  CK(h, cudaMemsetAsync(h->dev + F.off_zway, 0, (size_t)c.n_layers * c.max_seqs * c.n_kv_heads *
                        (std::max(c.k_cap, 1) + std::max(c.prefetch, 0)) * sizeof(uint2), h->main));
  CK(h, cudaMemsetAsync(h->dev + F.off_stats, 0, ST_COUNT * 8, h->main));
  CK(h, cudaMemsetAsync(h->dev + F.off_zoom_mask, 0, (size_t)regions * F.mask_words * 4, h->main));
  CK(h, cudaMemsetAsync(h->dev + F.off_zmask2, 0, (size_t)regions * F.mask_words * 8, h->main));      // stamps restart
  CK(h, cudaMemsetAsync(h->dev + F.off_err_flag, 0, 16, h->main));
  CK(h, cudaMemsetAsync(h->dev + F.off_ctrs, 0, (size_t)c.n_layers * F.ctrs_per_layer * 4, h->main));
  CK(h, cudaMemsetAsync(h->dev + F.off_plan_counts, 0, (size_t)regions * 2 * 4, h->main));
  CK(h, cudaStreamSynchronize(h->main));
  h->pending_prefetch = -1; h->pending_prefetch2 = -1;
  h->n_items = 0; h->use_fused = false; h->fused_why = "no sequences built";
  h->n_seqs = 0; h->segmented = false; h->m_b.clear(); h->A_b.clear(); h->tok_off.clear();
  h->span_len_host.clear();
  h->m_tot = h->A_tot = h->max_m = 0;
  h->layer_built.assign(c.n_layers, 0);
  h->host_used = 0;
  h->n_chunks = 0; h->parts1_max = 0; h->sort_n = 0;
  h->P2 = (std::max(c.k_cap, 1) + kStage2SpansPerCta - 1) / kStage2SpansPerCta;
  h->parts_per_head = 0;
  h->err.clear();
  return SEKV_OK;
}

sekv_status sekv_cache_flush(sekv_handle* h) {
  if (!h) return SEKV_INVALID_ARG;
  const sekv_config& c = h->cfg;
  const int64_t regions = (int64_t)c.n_layers * c.max_seqs * c.n_kv_heads;
  CK(h, cudaStreamSynchronize(h->side));
  CK(h, cudaMemsetAsync(h->dev + h->lay.cache_tags, 0xFF, regions * c.cache_ways * 4, h->main));
  CK(h, cudaMemsetAsync(h->dev + h->lay.cache_stamps, 0, regions * c.cache_ways * 4, h->main));
  return SEKV_OK;
}

// ---- build -------------------------------------------------------------------------------------------
static sekv_status make_schedule(sekv_handle* h) {
  // Static stage-1 schedule: entry rows of every (sequence, kv head) cut into near-equal chunks so
  // that the grid is ~ stage1_ctas CTAs of equal work (ragged contexts).
  const FullLayout& F = h->F;
  const sekv_config& c = h->cfg;
  const int B = h->n_seqs, Hkv = c.n_kv_heads;
  int target_ctas = c.stage1_ctas > 0 ? c.stage1_ctas : h->num_sms * 4;
  long total_tiles = 0;
  std::vector<int> tiles(B);
  for (int b = 0; b < B; ++b) {
    tiles[b] = (h->A_b[b] + h->m_b[b] + kTile - 1) / kTile;
    total_tiles += (long)tiles[b] * Hkv;
  }
  std::vector<Chunk> chunks;
  std::vector<int32_t> bg_begin(B * Hkv + 1, 0);
  int parts1_max = 0;
  for (int b = 0; b < B; ++b) {
    int rows = h->A_b[b] + h->m_b[b];
    int n = 0;
    if (rows > 0) {
      double share = total_tiles > 0 ? (double)tiles[b] * target_ctas / (double)total_tiles : 1.0;
      n = std::max(1, (int)std::floor(share + 0.5));
      n = std::min(n, tiles[b]);
    }
    for (int g = 0; g < Hkv; ++g) {
      bg_begin[b * Hkv + g] = (int32_t)chunks.size();
      if (n == 0) continue;
      int per = (tiles[b] + n - 1) / n;
      int part = 0;
      for (int t0 = 0; t0 < tiles[b]; t0 += per, ++part) {
        Chunk ck;
        ck.bg = b * Hkv + g;
        ck.row_begin = t0 * kTile;
        ck.row_end = std::min(rows, (t0 + per) * kTile);
        ck.part = part;
        chunks.push_back(ck);
      }
      parts1_max = std::max(parts1_max, part);
    }
  }
  bg_begin[B * Hkv] = (int32_t)chunks.size();
  if ((int)chunks.size() > F.max_chunks) return fail(h, SEKV_UNSUPPORTED, "stage-1 schedule exceeds chunk capacity");
  h->n_chunks = (int)chunks.size();
  h->parts1_max = parts1_max;
  h->parts_per_head = parts1_max + h->P2;
  if (!chunks.empty())
    CK(h, cudaMemcpyAsync(h->dev + F.off_chunks, chunks.data(), chunks.size() * sizeof(Chunk), cudaMemcpyHostToDevice, h->main));
  CK(h, cudaMemcpyAsync(h->dev + F.off_bg_chunk, bg_begin.data(), bg_begin.size() * 4, cudaMemcpyHostToDevice, h->main));
  CK(h, cudaStreamSynchronize(h->main));
  int sn = 32;
  while (sn < h->max_m) sn <<= 1;
  h->sort_n = sn;
  return SEKV_OK;
}

// Work-item list of the fused layer kernel (bf16 path), in queue order: POOL, COARSE, ZOOM, COMBINE -- a
// topological order of the dependencies (COARSE / ZOOM after the group's chain, which is not an item; COMBINE
// after the attention items).  When the batch does not fit the kernel (or impl = 1 / fp32 storage) the generic
// multi-kernel path runs instead and h->fused_why says why (sekv_get_path).
static sekv_status make_fused_schedule(sekv_handle* h) {
  const FullLayout& F = h->F;
  const sekv_config& c = h->cfg;
  h->use_fused = false;
  if (c.dtype != SEKV_BF16) { h->fused_why = "fp32 storage runs on the generic kernels"; return SEKV_OK; }
  if (c.impl == 1) { h->fused_why = "impl = 1 forces the generic kernels"; return SEKV_OK; }
  const int B = h->n_seqs, Hkv = c.n_kv_heads, BG = B * Hkv, G = h->G;
  if (c.route_dim != 8 && c.route_dim != 16 && c.route_dim != 32 && c.route_dim != 64) {
    h->fused_why = "route_dim is not 8, 16, 32 or 64"; return SEKV_OK;
  }
  if (!fused_geometry(h, nullptr, &h->fused_why)) return SEKV_OK;
  // the kernel spins on counters published by other CTAs: the whole grid must be resident (one CTA per SM)
  int per_sm = 0;
  cudaError_t oe = fused_occupancy(h, &per_sm);
  if (oe != cudaSuccess || per_sm < 1) {
    cudaGetLastError();
    h->fused_why = "the fused layer kernel cannot be resident on this device (shared memory / registers)";
    return SEKV_OK;
  }
  h->fused_grid = h->num_sms;
  FusedParams geo;
  fused_geometry(h, &geo, nullptr);
  const int n_chain_cta = std::min(BG, h->fused_grid);
  const int n_first = n_chain_cta * (fused_warps() - geo.team_warps) + (h->fused_grid - n_chain_cta) * fused_warps();
  // POOL items: by default sized so that ONE round over the warps that do not start on a chain covers every
  // pool row (they stream while the teams run the chains)
  // (the copies of the previous layer's prefetch candidates take first-round warps too: see the queue order below)
  const int n_pf = (c.k_cap > 0 && c.prefetch > 0 && c.n_layers > 1) ? BG * c.prefetch : 0;
  const int n_first_pool = n_first - n_pf > n_first / 2 ? n_first - n_pf : n_first;
  const bool pf_first = n_pf > 0 && n_first_pool < n_first;
  int rows = c.item_rows;
  if (rows <= 0) {
    long pool_rows = 0;
    for (int b = 0; b < B; ++b) pool_rows += (long)h->A_b[b] * Hkv;
    rows = (int)((pool_rows / std::max(n_first_pool, 1) + 1 + 15) / 16 * 16);
    rows = std::min(256, std::max(32, rows));
  }
  h->fused_item_rows = rows;
  const int crows = 32;        // COARSE items: two tiles, both in flight while the item waits for the zoom mask
  const int zs = 1;            // one expanded span per ZOOM item (zoom_spans_per_item is accepted and ignored)
  std::vector<Item> items;
  std::vector<int32_t> nparts(BG, 0), pbase(BG, 0);
  std::vector<int32_t> row0(B, 0), span0(B, 0);
  for (int b = 1; b < B; ++b) { row0[b] = row0[b - 1] + h->A_b[b - 1] + h->m_b[b - 1]; span0[b] = span0[b - 1] + h->m_b[b - 1]; }
  auto mk = [&](int kind, int b, int g, int a, int bb, int part) {
    Item it;
    memset(&it, 0, sizeof(it));
    it.kind = kind; it.bg = b * Hkv + g; it.a = a; it.b = bb; it.part = part;
    it.A = h->A_b[b]; it.row0 = row0[b]; it.span0 = span0[b];
    return it;
  };
  // partial slots first (attention items need np of their group)
  for (int b = 0; b < B; ++b)
    for (int g = 0; g < Hkv; ++g) {
      const int A = h->A_b[b], m = h->m_b[b];
      int n = (A + rows - 1) / rows + (m + crows - 1) / crows;
      if (c.k_cap > 0) n += (std::min(c.k_cap, m) + zs - 1) / zs;
      nparts[b * Hkv + g] = n;
    }
  int total_parts = 0;
  for (int bg = 0; bg < BG; ++bg) { pbase[bg] = total_parts * G; total_parts += nparts[bg]; }
  if (total_parts > F.max_chunks) { h->fused_why = "partial-record table too small for this batch"; return SEKV_OK; }
  std::vector<int32_t> next_part(BG, 0);
  auto attn = [&](std::vector<Item>& dst, int kind, int b, int g, int a, int bb) {
    const int bg = b * Hkv + g;
    Item it = mk(kind, b, g, a, bb, next_part[bg]++);
    it.pbase = pbase[bg]; it.np = nparts[bg];
    dst.push_back(it);
  };
  // Queue order: [POOL: one item for every warp that does not start on a chain] [ZOOM] [COARSE] [rest of POOL]
  // [COMBINE].  The first round of POOL items streams while the teams run the chains; the items that wait for a
  // chain (latency-bound ZOOM first) follow, and the remaining dependency-free POOL rows fill the tail.
  // (partial slots of a group: POOL, then COARSE, then ZOOM -- COMBINE merges the first two kinds early)
  std::vector<Item> pool_items, coarse_items, zoom_items;
  for (int b = 0; b < B; ++b)
    for (int g = 0; g < Hkv; ++g)
      for (int r0 = 0; r0 < h->A_b[b]; r0 += rows) attn(pool_items, IT_POOL, b, g, r0, std::min(h->A_b[b], r0 + rows));
  for (int b = 0; b < B; ++b)
    for (int g = 0; g < Hkv; ++g) {
      const int A = h->A_b[b], R = A + h->m_b[b];
      for (int r0 = A; r0 < R; r0 += crows) attn(coarse_items, IT_COARSE, b, g, r0, std::min(R, r0 + crows));
    }
  if (c.k_cap > 0)
    for (int b = 0; b < B; ++b)
      for (int g = 0; g < Hkv; ++g) {
        const int kmax = std::min(c.k_cap, h->m_b[b]);
        for (int j0 = 0; j0 < kmax; j0 += zs) attn(zoom_items, IT_ZOOM, b, g, j0, std::min(kmax, j0 + zs));
      }
  // Prefetch candidates of the previous layer of the step (copied by this layer's kernel; mostly no-ops).  Their
  // blobs cross PCIe, and so do the demand misses of THIS layer, which are known only once its chains have run: the
  // copies go out first (spread over the first round, so that no SM is left without POOL rows to stream) and the
  // link is free again when the demand misses arrive.
  std::vector<Item> pf_items;
  if (n_pf > 0)
    for (int i = 0; i < c.prefetch; ++i)
      for (int b = 0; b < B; ++b)
        for (int g = 0; g < Hkv; ++g) pf_items.push_back(mk(IT_PREFETCH, b, g, i, 0, 0));
  const size_t first = std::min<size_t>((size_t)std::max(pf_first ? n_first_pool : n_first, 0), pool_items.size());
  if (pf_first) {
    const size_t total = first + pf_items.size();
    size_t ip = 0, ipf = 0;
    for (size_t i = 0; i < total; ++i) {
      // slot i takes a copy when the copies are behind their even share
      if (ipf < pf_items.size() && (ip >= first || ipf * total <= i * pf_items.size())) items.push_back(pf_items[ipf++]);
      else items.push_back(pool_items[ip++]);
    }
  } else {
    items.insert(items.end(), pool_items.begin(), pool_items.begin() + first);
    items.insert(items.end(), pf_items.begin(), pf_items.end());
  }
  h->pool_end = (int)items.size();
  // ZOOM positions 0 and 1 of every group first (the plan puts demand misses there: their blobs cross PCIe), then
  // the COARSE items (two tiles each, in flight while the item waits for the zoom mask; ~1 us of work after it),
  // then the other ZOOM items
  std::vector<Item> zoom_early, zoom_late;
  for (const Item& it : zoom_items) (it.a < 2 ? zoom_early : zoom_late).push_back(it);
  items.insert(items.end(), zoom_early.begin(), zoom_early.end());
  items.insert(items.end(), coarse_items.begin(), coarse_items.end());
  items.insert(items.end(), zoom_late.begin(), zoom_late.end());
  items.insert(items.end(), pool_items.begin() + first, pool_items.end());
  for (int b = 0; b < B; ++b)
    for (int g = 0; g < Hkv; ++g)
      for (int hl = 0; hl < G; ++hl) {
        Item it = mk(IT_COMBINE, b, g, hl, (h->A_b[b] + rows - 1) / rows + (h->m_b[b] + crows - 1) / crows, 0);   // b = POOL + COARSE partials
        it.pbase = pbase[b * Hkv + g]; it.np = nparts[b * Hkv + g];
        items.push_back(it);
      }
  if ((int)items.size() > F.max_items) { h->fused_why = "work-item table too small for this batch"; return SEKV_OK; }
  h->n_items = (int)items.size();
  std::vector<int32_t> grp((size_t)BG * 2);
  for (int b = 0; b < B; ++b)
    for (int g = 0; g < Hkv; ++g) { grp[2 * (b * Hkv + g)] = span0[b]; grp[2 * (b * Hkv + g) + 1] = h->m_b[b]; }
  CK(h, cudaMemcpyAsync(h->dev + F.off_bg_part, grp.data(), grp.size() * 4, cudaMemcpyHostToDevice, h->main));
  CK(h, cudaMemcpyAsync(h->dev + F.off_items_sched, items.data(), items.size() * sizeof(Item), cudaMemcpyHostToDevice, h->main));
  CK(h, cudaStreamSynchronize(h->main));
  h->use_fused = true;
  h->fused_why.clear();
  return SEKV_OK;
}

static sekv_status ensure_segmented(sekv_handle* h, int n_seqs, const int64_t* seq_tok_off, const float* H) {
  const sekv_config& c = h->cfg;
  if (n_seqs < 1 || n_seqs > c.max_seqs) return fail(h, SEKV_INVALID_ARG, "n_seqs out of range");
  if (!seq_tok_off) return fail(h, SEKV_INVALID_ARG, "seq_tok_off is NULL");
  if (seq_tok_off[0] != 0) return fail(h, SEKV_INVALID_ARG, "seq_tok_off[0] != 0");
  for (int b = 0; b < n_seqs; ++b)
    if (seq_tok_off[b + 1] <= seq_tok_off[b]) return fail(h, SEKV_INVALID_ARG, "empty or negative-length sequence");
  if (seq_tok_off[n_seqs] > c.max_tokens_total) return fail(h, SEKV_OOM_DEVICE, "sum of tokens exceeds max_tokens_total");
  if (h->segmented) {
    if (n_seqs != h->n_seqs) return fail(h, SEKV_STATE, "batch size differs from the segmented batch");
    for (int b = 0; b <= n_seqs; ++b)
      if (seq_tok_off[b] != h->tok_off[b]) return fail(h, SEKV_STATE, "token offsets differ from the segmented batch");
    return SEKV_OK;
  }
  if (!H) return fail(h, SEKV_INVALID_ARG, "H is NULL on the first build call");
  std::vector<int> m(n_seqs), a(n_seqs);
  std::string why;
  h->n_seqs = n_seqs;
  cudaError_t e = launch_segment(h, H, n_seqs, seq_tok_off, m.data(), a.data(), &why);
  if (e != cudaSuccess) { h->n_seqs = 0; return cuda_fail(h, e, "segmentation"); }
  if (!why.empty()) { h->n_seqs = 0; return fail(h, why.find("capacity") != std::string::npos ? SEKV_OOM_DEVICE : SEKV_UNSUPPORTED, why); }
  h->m_b = m; h->A_b = a;
  h->tok_off.assign(seq_tok_off, seq_tok_off + n_seqs + 1);
  h->m_tot = 0; h->A_tot = 0; h->max_m = 0;
  for (int b = 0; b < n_seqs; ++b) { h->m_tot += m[b]; h->A_tot += a[b]; h->max_m = std::max(h->max_m, m[b]); }
  h->segmented = true;
  sekv_status ss = make_schedule(h);
  if (ss != SEKV_OK) return ss;
  return make_fused_schedule(h);
}

static sekv_status assign_blobs(sekv_handle* h, int layer, const std::vector<int32_t>& rk, const std::vector<int32_t>& rv) {
  // rk, rv: [H_kv][m_tot] retained ranks (host copies).  Bump-allocates the host arena.
  const sekv_config& c = h->cfg;
  const int Hkv = c.n_kv_heads, m = h->m_tot;
  std::vector<int64_t> off((size_t)Hkv * h->lay.spans_cap, 0);
  std::vector<int32_t> rank((size_t)Hkv * h->lay.spans_cap, 0);
  size_t used = round_up_sz(h->host_used, 128);
  for (int g = 0; g < Hkv; ++g)
    for (int s = 0; s < m; ++s) {
      int len = h->span_len_host[s];
      int a = rk[(size_t)g * m + s], b = rv[(size_t)g * m + s];
      if (a < 0 || b < 0 || a > c.r_max || b > c.r_max || a > len || b > len)
        return fail(h, SEKV_INVALID_ARG, "retained rank out of range (must be <= min(r_max, |S|))");
      BlobDims bd = blob_dims(h->esize, len, a, b);
      off[(size_t)g * h->lay.spans_cap + s] = (int64_t)used;
      rank[(size_t)g * h->lay.spans_cap + s] = a | (b << 8) | (len << 16);   // the fused kernel's span meta word
      used += bd.bytes;
    }
  if (used > h->host_bytes) return fail(h, SEKV_OOM_HOST, "pinned host arena too small for the factor store");
  LayerView lv = layer_view(h, layer);
  CK(h, cudaMemcpyAsync((void*)lv.dir_off, off.data(), off.size() * 8, cudaMemcpyHostToDevice, h->main));
  CK(h, cudaMemcpyAsync((void*)lv.dir_rank, rank.data(), rank.size() * 4, cudaMemcpyHostToDevice, h->main));
  CK(h, cudaStreamSynchronize(h->main));
  h->host_used = used;
  return SEKV_OK;
}

static void report_counts(sekv_handle* h, int32_t* spans_per_seq, int32_t* pool_per_seq) {
  for (int b = 0; b < h->n_seqs; ++b) {
    if (spans_per_seq) spans_per_seq[b] = h->m_b[b];
    if (pool_per_seq) pool_per_seq[b] = h->A_b[b];
  }
}

sekv_status sekv_build_spans_prefactored(sekv_handle* h, int32_t layer, int32_t n_seqs, const int64_t* seq_tok_off,
                                         const float* H, const sekv_factors* f, const void* W,
                                         int32_t* spans_per_seq, int32_t* pool_per_seq) {
  if (!h) return SEKV_INVALID_ARG;
  const sekv_config& c = h->cfg;
  if (layer < 0 || layer >= c.n_layers) return fail(h, SEKV_INVALID_ARG, "layer out of range");
  if (!f || !W) return fail(h, SEKV_INVALID_ARG, "factors or W is NULL");
  if (f->rank_in < 1 || f->rank_in > SEKV_MAX_RANK) return fail(h, SEKV_INVALID_ARG, "rank_in out of range");
  if (!f->tokUK || !f->SK || !f->VtK || !f->tokUV || !f->SV || !f->VtV) return fail(h, SEKV_INVALID_ARG, "NULL factor array");
  if (!H) return fail(h, SEKV_INVALID_ARG, "H is NULL (the summaries need the surprisal weights)");
  sekv_status s = ensure_segmented(h, n_seqs, seq_tok_off, H);
  if (s != SEKV_OK) return s;
  if (f->m_tot != h->m_tot || f->a_tot != h->A_tot) {
    char buf[160];
    snprintf(buf, sizeof(buf), "segmentation found m_tot=%d A_tot=%d but the factors were laid out for m_tot=%d A_tot=%d",
             h->m_tot, h->A_tot, f->m_tot, f->a_tot);
    return fail(h, SEKV_STATE, buf);
  }
  if (h->A_tot > 0 && (!f->Kfull || !f->Vfull)) return fail(h, SEKV_INVALID_ARG, "Kfull/Vfull is NULL");
  const int Hkv = c.n_kv_heads, m = h->m_tot;
  std::vector<int32_t> rk((size_t)Hkv * m), rv((size_t)Hkv * m);
  if (f->rank_k) CK(h, cudaMemcpy(rk.data(), f->rank_k, rk.size() * 4, cudaMemcpyDeviceToHost));
  if (f->rank_v) CK(h, cudaMemcpy(rv.data(), f->rank_v, rv.size() * 4, cudaMemcpyDeviceToHost));
  for (int g = 0; g < Hkv; ++g)
    for (int sidx = 0; sidx < m; ++sidx) {
      int cap = std::min({(int)f->rank_in, h->span_len_host[sidx], c.r_max});
      if (!f->rank_k) rk[(size_t)g * m + sidx] = cap;
      if (!f->rank_v) rv[(size_t)g * m + sidx] = cap;
      if (rk[(size_t)g * m + sidx] > f->rank_in || rv[(size_t)g * m + sidx] > f->rank_in)
        return fail(h, SEKV_INVALID_ARG, "retained rank exceeds rank_in");
    }
  s = assign_blobs(h, layer, rk, rv);
  if (s != SEKV_OK) return s;
  cudaError_t e = launch_build_prefactored(h, layer, H, f, W);
  if (e != cudaSuccess) return cuda_fail(h, e, "build (prefactored)");
  CK(h, cudaStreamSynchronize(h->main));
  h->layer_built[layer] = 1;
  report_counts(h, spans_per_seq, pool_per_seq);
  return SEKV_OK;
}

sekv_status sekv_build_spans(sekv_handle* h, int32_t layer, int32_t n_seqs, const int64_t* seq_tok_off,
                             const float* H, const void* K, const void* V, const void* W, int32_t rank_cap,
                             int32_t* spans_per_seq, int32_t* pool_per_seq) {
  if (!h) return SEKV_INVALID_ARG;
  const sekv_config& c = h->cfg;
  if (layer < 0 || layer >= c.n_layers) return fail(h, SEKV_INVALID_ARG, "layer out of range");
  if (!K || !V || !W) return fail(h, SEKV_INVALID_ARG, "K, V or W is NULL");
  if (!H) return fail(h, SEKV_INVALID_ARG, "H is NULL (the summaries need the surprisal weights)");
  if (rank_cap < 0 || rank_cap > c.r_max) return fail(h, SEKV_INVALID_ARG, "rank_cap out of range");
  if (rank_cap == 0) rank_cap = c.r_max;
  sekv_status s = ensure_segmented(h, n_seqs, seq_tok_off, H);
  if (s != SEKV_OK) return s;
  const int Hkv = c.n_kv_heads, m = h->m_tot;
  std::vector<int32_t> rk((size_t)Hkv * m), rv;
  for (int g = 0; g < Hkv; ++g)
    for (int sidx = 0; sidx < m; ++sidx)
      rk[(size_t)g * m + sidx] = std::min({rank_cap, h->span_len_host[sidx], (int)kD});   // Eq. 6: R = min(|S|, d_h, R_max)
  rv = rk;
  s = assign_blobs(h, layer, rk, rv);
  if (s != SEKV_OK) return s;
  std::string why;
  cudaError_t e = launch_build_dense(h, layer, H, K, V, W, rank_cap, &why);
  if (e != cudaSuccess) return cuda_fail(h, e, "build (dense)");
  if (!why.empty()) return fail(h, SEKV_UNSUPPORTED, why);
  CK(h, cudaStreamSynchronize(h->main));
  h->layer_built[layer] = 1;
  report_counts(h, spans_per_seq, pool_per_seq);
  return SEKV_OK;
}

// ---- decode --------------------------------------------------------------------------------------------
// CUDA-event bracket around one kernel launch when profiling is on (never during graph capture)
struct ProfScope {
  sekv_handle* h; cudaStream_t s; int idx;
  ProfScope(sekv_handle* h_, int cls, cudaStream_t s_) : h(h_), s(s_), idx(-1) {
    if (!h->profiling) return;
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(s, &st) != cudaSuccess || st != cudaStreamCaptureStatusNone) return;
    sekv_handle::ProfRec r;
    r.cls = cls;
    if (cudaEventCreate(&r.a) != cudaSuccess) return;
    if (cudaEventCreate(&r.b) != cudaSuccess) { cudaEventDestroy(r.a); return; }
    cudaEventRecord(r.a, s);
    h->prof.push_back(r);
    idx = (int)h->prof.size() - 1;
  }
  ~ProfScope() { if (idx >= 0) cudaEventRecord(h->prof[idx].b, s); }
};

static sekv_status check_ready(sekv_handle* h, int layer) {
  if (!h->segmented) return fail(h, SEKV_STATE, "no sequences built");
  if (layer < 0 || layer >= h->cfg.n_layers) return fail(h, SEKV_INVALID_ARG, "layer out of range");
  if (!h->layer_built[layer]) return fail(h, SEKV_STATE, "layer not built");
  return SEKV_OK;
}

static sekv_status check_k(sekv_handle* h, int k) {
  if (k > h->cfg.k_cap) return fail(h, SEKV_INVALID_ARG, "k exceeds k_cap");
  if (k < 0 && h->max_m > h->cfg.k_cap) return fail(h, SEKV_INVALID_ARG, "k < 0 (all spans) needs k_cap >= spans per sequence");
  return SEKV_OK;
}

sekv_status sekv_route(sekv_handle* h, int32_t layer, const void* q, const float* tau, int32_t k, float* logits,
                       float* alpha_tilde, int32_t* ids, int32_t* count) {
  if (!h) return SEKV_INVALID_ARG;
  sekv_status s = check_ready(h, layer);
  if (s != SEKV_OK) return s;
  if (!q || !ids || !count) return fail(h, SEKV_INVALID_ARG, "q, ids or count is NULL");
  if ((s = check_k(h, k)) != SEKV_OK) return s;
  cudaError_t e;
  if (h->use_fused) {
    ProfScope ps(h, 6, h->main);
    e = launch_fused(h, layer, FM_ROUTE, q, tau, k, logits, alpha_tilde, ids, count, nullptr, nullptr, h->main);
  } else {
    ProfScope ps(h, 0, h->main);
    e = launch_route(h, layer, q, tau, k, logits, alpha_tilde, ids, count, h->main);
  }
  if (e != cudaSuccess) return cuda_fail(h, e, "route");
  return SEKV_OK;
}

static cudaError_t decode_layer(sekv_handle* h, int layer, const void* q, const int32_t* ids, const int32_t* count,
                                void* out, float* lse) {
  cudaError_t e;
  if (h->use_fused) {     // caller-supplied zoom set: plan + attention + combine in the fused layer kernel
    if (h->pending_prefetch == layer || h->pending_prefetch2 == layer) {   // this layer's cache is about to be read: finish its prefetch copies first
      if ((e = launch_prefetch(h, layer, h->main)) != cudaSuccess) return e;
      if (h->pending_prefetch == layer) h->pending_prefetch = -1; else h->pending_prefetch2 = -1;
    }
    ProfScope ps(h, 6, h->main);
    return launch_fused(h, layer, FM_ATTN, q, nullptr, 0, nullptr, nullptr, (int32_t*)ids, (int32_t*)count, out, lse, h->main);
  }
  { ProfScope ps(h, 1, h->main); if ((e = launch_plan(h, layer, ids, count, h->main)) != cudaSuccess) return e; }
  if (h->cfg.k_cap > 0) {
    if ((e = cudaEventRecord(h->ev_fork, h->main)) != cudaSuccess) return e;
    if ((e = cudaStreamWaitEvent(h->side, h->ev_fork, 0)) != cudaSuccess) return e;
    { ProfScope ps(h, 2, h->side); if ((e = launch_fetch(h, layer, count, h->side)) != cudaSuccess) return e; }
    if ((e = cudaEventRecord(h->ev_join, h->side)) != cudaSuccess) return e;
  }
  { ProfScope ps(h, 3, h->main); if ((e = launch_stage1(h, layer, q, h->main)) != cudaSuccess) return e; }
  if (h->cfg.k_cap > 0) {
    if ((e = cudaStreamWaitEvent(h->main, h->ev_join, 0)) != cudaSuccess) return e;
    ProfScope ps(h, 4, h->main);
    if ((e = launch_stage2(h, layer, q, count, h->main)) != cudaSuccess) return e;
  }
  ProfScope ps(h, 5, h->main);
  return launch_combine(h, layer, out, lse, h->main);
}

sekv_status sekv_decode_attn(sekv_handle* h, int32_t layer, const void* q, const int32_t* ids, const int32_t* count,
                             void* out, float* lse) {
  if (!h) return SEKV_INVALID_ARG;
  sekv_status s = check_ready(h, layer);
  if (s != SEKV_OK) return s;
  if (!q || !out) return fail(h, SEKV_INVALID_ARG, "q or out is NULL");
  if (h->cfg.k_cap > 0 && (!ids || !count)) return fail(h, SEKV_INVALID_ARG, "ids or count is NULL");
  cudaError_t e = decode_layer(h, layer, q, ids, count, out, lse);
  if (e != cudaSuccess) return cuda_fail(h, e, "decode_attn");
  return SEKV_OK;
}

static cudaError_t enqueue_step(sekv_handle* h, const void* q, const float* tau, int k, void* out, float* lse) {
  const sekv_config& c = h->cfg;
  const int B = h->n_seqs;
  const size_t qstride = (size_t)B * c.n_q_heads * kD * h->esize;
  const size_t ostride = (size_t)B * c.n_q_heads * kD * (c.out_dtype == SEKV_BF16 ? 2 : 4);
  const int kcap = std::max(c.k_cap, 1);
  for (int l = 0; l < c.n_layers; ++l) {
    const uint8_t* ql = (const uint8_t*)q + l * qstride;
    int32_t* ids = (int32_t*)(h->dev + h->F.off_ws_ids) + (size_t)l * c.max_seqs * c.n_kv_heads * kcap;
    int32_t* cnt = (int32_t*)(h->dev + h->F.off_ws_count) + (size_t)l * c.max_seqs * c.n_kv_heads;
    cudaError_t e;
    void* ol = (uint8_t*)out + l * ostride;
    float* ll = lse ? lse + (size_t)l * B * c.n_q_heads : nullptr;
    if (h->use_fused) {
      if (c.n_layers == 1 && c.k_cap > 0 && c.prefetch > 0) {
        // a one-layer model has no following layer kernel to carry the copies of the previous step's candidates
        ProfScope ps(h, 7, h->main);
        if ((e = launch_prefetch(h, 0, h->main)) != cudaSuccess) return e;
      }
      {
        ProfScope ps(h, 6, h->main);
        if (c.k_cap > 0)
          e = launch_fused(h, l, FM_ROUTE | FM_ATTN, ql, tau ? tau + (size_t)l * c.n_q_heads : nullptr, k, nullptr,
                           nullptr, ids, cnt, ol, ll, h->main);
        else
          e = launch_fused(h, l, FM_ATTN, ql, nullptr, 0, nullptr, nullptr, nullptr, nullptr, ol, ll, h->main);
      }
      if (e != cudaSuccess) return e;
      continue;
    }
    if (c.k_cap > 0) {
      ProfScope ps(h, 0, h->main);
      e = launch_route(h, l, ql, tau ? tau + (size_t)l * c.n_q_heads : nullptr, k, nullptr, nullptr, ids, cnt, h->main);
      if (e != cudaSuccess) return e;
    }
    e = decode_layer(h, l, ql, ids, cnt, ol, ll);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

static sekv_status decode_step_impl(sekv_handle* h, const void* q, const float* tau, int32_t k, void* out, float* lse) {
  if (!h) return SEKV_INVALID_ARG;
  if (!h->segmented) return fail(h, SEKV_STATE, "no sequences built");
  for (int l = 0; l < h->cfg.n_layers; ++l)
    if (!h->layer_built[l]) return fail(h, SEKV_STATE, "not every layer is built");
  if (!q || !out) return fail(h, SEKV_INVALID_ARG, "q or out is NULL");
  sekv_status s = check_k(h, k);
  if (s != SEKV_OK) return s;
  if (!h->cfg.use_graph || h->profiling) {   // profiling brackets kernels with events: eager launches only
    cudaError_t e = enqueue_step(h, q, tau, k, out, lse);
    if (e != cudaSuccess) return cuda_fail(h, e, "decode_step");
    return SEKV_OK;
  }
  for (auto& g : h->graphs)
    if (g.q == q && g.tau == tau && g.k == k && g.out == out && g.lse == lse) {
      CK(h, cudaGraphLaunch(g.exec, h->main));
      h->launches += g.nodes;
      return SEKV_OK;
    }
  // capture once for this argument tuple
  uint64_t before = h->launches;
  CK(h, cudaStreamBeginCapture(h->main, cudaStreamCaptureModeRelaxed));
  cudaError_t e = enqueue_step(h, q, tau, k, out, lse);
  cudaGraph_t graph = nullptr;
  cudaError_t e2 = cudaStreamEndCapture(h->main, &graph);
  uint64_t nodes = h->launches - before;
  h->launches = before;
  if (e != cudaSuccess || e2 != cudaSuccess) {
    if (graph) cudaGraphDestroy(graph);
    cudaGetLastError();
    if (h->use_pdl) { h->use_pdl = false; return decode_step_impl(h, q, tau, k, out, lse); }   // retry without the PDL edges
    return cuda_fail(h, e != cudaSuccess ? e : e2, "decode_step graph capture");
  }
  GraphEntry ge{q, tau, k, out, lse, nullptr, nodes};
  cudaError_t e3 = cudaGraphInstantiate(&ge.exec, graph, 0);
  cudaGraphDestroy(graph);
  if (e3 != cudaSuccess) {
    cudaGetLastError();
    if (h->use_pdl) { h->use_pdl = false; return decode_step_impl(h, q, tau, k, out, lse); }
    return cuda_fail(h, e3, "cudaGraphInstantiate");
  }
  if (h->graphs.size() >= 64) { cudaGraphExecDestroy(h->graphs.front().exec); h->graphs.erase(h->graphs.begin()); }
  h->graphs.push_back(ge);
  CK(h, cudaGraphLaunch(ge.exec, h->main));
  h->launches += nodes;
  return SEKV_OK;
}

sekv_status sekv_decode_step(sekv_handle* h, const void* q, const float* tau, int32_t k, void* out, float* lse) {
  const sekv_status s = decode_step_impl(h, q, tau, k, out, lse);
  // the last layer's prefetch candidates are copied by layer 0 of the next step (or before the next read of its cache)
  if (s == SEKV_OK && h->use_fused && h->cfg.k_cap > 0 && h->cfg.prefetch > 0 && k >= 0) {
    h->pending_prefetch = h->cfg.n_layers - 1;
    // (three layers or more: a layer's candidates are copied two launches later, fused_kernels.cu)
    h->pending_prefetch2 = h->cfg.n_layers >= 3 ? h->cfg.n_layers - 2 : -1;
  }
  return s;
}

sekv_status sekv_last_zoom_ids(sekv_handle* h, int32_t layer, int32_t* ids, int32_t* count) {
  if (!h) return SEKV_INVALID_ARG;
  sekv_status s = check_ready(h, layer);
  if (s != SEKV_OK) return s;
  if (!ids || !count) return fail(h, SEKV_INVALID_ARG, "ids or count is NULL");
  const sekv_config& c = h->cfg;
  const int kcap = std::max(c.k_cap, 1);
  const int32_t* wi = (const int32_t*)(h->dev + h->F.off_ws_ids) + (size_t)layer * c.max_seqs * c.n_kv_heads * kcap;
  const int32_t* wc = (const int32_t*)(h->dev + h->F.off_ws_count) + (size_t)layer * c.max_seqs * c.n_kv_heads;
  CK(h, cudaMemcpyAsync(ids, wi, (size_t)h->n_seqs * c.n_kv_heads * kcap * 4, cudaMemcpyDeviceToDevice, h->main));
  CK(h, cudaMemcpyAsync(count, wc, (size_t)h->n_seqs * c.n_kv_heads * 4, cudaMemcpyDeviceToDevice, h->main));
  return SEKV_OK;
}

sekv_status sekv_decode_step_host(sekv_handle* h, const void* q_host, const float* tau, int32_t k, void* out_host,
                                  float* lse_host) {
  if (!h) return SEKV_INVALID_ARG;
  if (!q_host || !out_host) return fail(h, SEKV_INVALID_ARG, "q_host or out_host is NULL");
  if (!h->segmented) return fail(h, SEKV_STATE, "no sequences built");
  const sekv_config& c = h->cfg;
  const size_t n = (size_t)c.n_layers * h->n_seqs * c.n_q_heads;
  void* qd = h->dev + h->F.off_q_stage;
  void* od = h->dev + h->F.off_out_stage;
  float* ld = (float*)(h->dev + h->F.off_lse_stage);
  CK(h, cudaMemcpyAsync(qd, q_host, n * kD * h->esize, cudaMemcpyHostToDevice, h->main));
  sekv_status s = sekv_decode_step(h, qd, tau, k, od, lse_host ? ld : nullptr);
  if (s != SEKV_OK) return s;
  CK(h, cudaMemcpyAsync(out_host, od, n * kD * (c.out_dtype == SEKV_BF16 ? 2 : 4), cudaMemcpyDeviceToHost, h->main));
  if (lse_host) CK(h, cudaMemcpyAsync(lse_host, ld, n * 4, cudaMemcpyDeviceToHost, h->main));
  CK(h, cudaStreamSynchronize(h->main));
  return SEKV_OK;
}

// ---- introspection ----------------------------------------------------------------------------------------
sekv_status sekv_get_layout(const sekv_handle* h, sekv_layout* out) {
  if (!h || !out) return SEKV_INVALID_ARG;
  *out = h->lay;
  out->host_bytes_used = (int64_t)h->host_used;
  return SEKV_OK;
}

sekv_status sekv_get_stats(sekv_handle* h, sekv_stats* out) {
  if (!h || !out) return SEKV_INVALID_ARG;
  CK(h, cudaStreamSynchronize(h->main));
  CK(h, cudaStreamSynchronize(h->side));
  uint64_t v[ST_COUNT];
  CK(h, cudaMemcpy(v, h->dev + h->F.off_stats, sizeof(v), cudaMemcpyDeviceToHost));
  out->layer_steps = v[ST_LAYER_STEPS];
  out->zoomed_spans = v[ST_ZOOMED];
  out->cache_hits = v[ST_HITS];
  out->cache_misses = v[ST_MISSES];
  out->h2d_bytes = v[ST_H2D];
  out->factor_bytes_algo = v[ST_FACTOR_ALGO];
  out->coarse_rows_skipped = v[ST_SKIPPED];
  out->prefetched_spans = v[ST_PREFETCHED];
  out->kernel_launches = h->launches;
  out->prefetch_h2d_bytes = v[ST_PF_BYTES];
  return SEKV_OK;
}

sekv_status sekv_reset_stats(sekv_handle* h) {
  if (!h) return SEKV_INVALID_ARG;
  CK(h, cudaMemsetAsync(h->dev + h->F.off_stats, 0, ST_COUNT * 8, h->main));
  h->launches = 0;
  return SEKV_OK;
}

sekv_status sekv_static_bytes_per_layer(const sekv_handle* h, uint64_t* bytes) {
  if (!h || !bytes) return SEKV_INVALID_ARG;
  const sekv_config& c = h->cfg;
  const uint64_t b = h->esize, bo = c.out_dtype == SEKV_BF16 ? 2 : 4;
  uint64_t t = (uint64_t)c.n_q_heads * c.route_dim * kD * b;   // W, once per layer
  for (int s = 0; s < h->n_seqs; ++s) {
    const uint64_t m = h->m_b[s], a = h->A_b[s];
    t += (uint64_t)c.n_q_heads * m * c.route_dim * b + 4 * m;   // routing summaries + ln|S|
    t += 2ull * c.n_kv_heads * a * kD * b;                      // pool K and V
    t += 2ull * c.n_kv_heads * m * kD * b;                      // coarse means (all; skipped rows subtracted via stats)
    t += (uint64_t)c.n_q_heads * kD * (b + bo);                 // q and out
  }
  *bytes = t;
  return SEKV_OK;
}

static void prof_clear(sekv_handle* h) {
  for (auto& r : h->prof) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
  h->prof.clear();
}

sekv_status sekv_set_profiling(sekv_handle* h, int32_t on) {
  if (!h) return SEKV_INVALID_ARG;
  h->profiling = on != 0;
  return SEKV_OK;
}

sekv_status sekv_get_kernel_times(sekv_handle* h, double* ms, uint64_t* launches) {
  if (!h || !ms || !launches) return SEKV_INVALID_ARG;
  CK(h, cudaStreamSynchronize(h->main));
  CK(h, cudaStreamSynchronize(h->side));
  for (int i = 0; i < SEKV_N_KERNEL_CLASSES; ++i) { ms[i] = 0.0; launches[i] = 0; }
  for (auto& r : h->prof) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, r.a, r.b) == cudaSuccess) { ms[r.cls] += t; launches[r.cls] += 1; }
  }
  cudaGetLastError();
  prof_clear(h);
  return SEKV_OK;
}

sekv_status sekv_set_trace(sekv_handle* h, void* buf, int64_t capacity_items, int32_t* n_items) {
  if (!h) return SEKV_INVALID_ARG;
  CK(h, cudaStreamSynchronize(h->main));
  h->trace_buf = buf;
  h->trace_cap = buf ? capacity_items : 0;
  for (auto& g : h->graphs) cudaGraphExecDestroy(g.exec);     // captured launches carry the old pointer
  h->graphs.clear();
  if (n_items) *n_items = h->n_items;
  return SEKV_OK;
}

sekv_status sekv_graph_count(const sekv_handle* h, int32_t* count) {
  if (!h || !count) return SEKV_INVALID_ARG;
  *count = (int32_t)h->graphs.size();
  return SEKV_OK;
}

sekv_status sekv_get_path(const sekv_handle* h, int32_t* fused, const char** reason) {
  if (!h) return SEKV_INVALID_ARG;
  if (fused) *fused = h->use_fused ? 1 : 0;
  if (reason) *reason = h->fused_why.c_str();
  return SEKV_OK;
}

sekv_status sekv_export_span_factors(sekv_handle* h, int32_t layer, int32_t seq, int32_t kv_head, int32_t span,
                                     int32_t* len_out, int32_t* rank_k, int32_t* rank_v, float* UK, float* sK,
                                     float* VtK, float* UV, float* sV, float* VtV, int32_t* pad_zero) {
  if (!h) return SEKV_INVALID_ARG;
  sekv_status s = check_ready(h, layer);
  if (s != SEKV_OK) return s;
  const sekv_config& c = h->cfg;
  if (seq < 0 || seq >= h->n_seqs || kv_head < 0 || kv_head >= c.n_kv_heads) return fail(h, SEKV_INVALID_ARG, "sequence or kv head out of range");
  if (span < 0 || span >= h->m_b[seq]) return fail(h, SEKV_INVALID_ARG, "span out of range");
  int gs = span;
  for (int b = 0; b < seq; ++b) gs += h->m_b[b];
  LayerView lv = layer_view(h, layer);
  int64_t off = 0;
  int32_t rr = 0;
  CK(h, cudaStreamSynchronize(h->main));
  CK(h, cudaMemcpy(&off, lv.dir_off + (size_t)kv_head * h->lay.spans_cap + gs, 8, cudaMemcpyDeviceToHost));
  CK(h, cudaMemcpy(&rr, lv.dir_rank + (size_t)kv_head * h->lay.spans_cap + gs, 4, cudaMemcpyDeviceToHost));
  const int len = h->span_len_host[gs], rk = rr & 0xff, rv = (rr >> 8) & 0xff, es = h->esize;
  if (len_out) *len_out = len;
  if (rank_k) *rank_k = rk;
  if (rank_v) *rank_v = rv;
  const BlobDims bd = blob_dims(es, len, rk, rv);
  const uint8_t* blob = h->host + off;
  auto ld = [&](size_t o) -> float {
    if (es == 4) { float v; memcpy(&v, blob + o, 4); return v; }
    uint16_t u; memcpy(&u, blob + o, 2);
    uint32_t w = (uint32_t)u << 16; float v; memcpy(&v, &w, 4); return v;
  };
  const float* bsk = (const float*)(blob + bd.off_sk);
  const float* bsv = (const float*)(blob + bd.off_sv);
  if (sK) for (int i = 0; i < rk; ++i) sK[i] = bsk[i];
  if (sV) for (int i = 0; i < rv; ++i) sV[i] = bsv[i];
  if (VtK) for (int i = 0; i < rk; ++i) for (int d = 0; d < kD; ++d) VtK[(size_t)i * kD + d] = ld(blob_vtk_off(bd, es, i, d));
  if (VtV) for (int i = 0; i < rv; ++i) for (int d = 0; d < kD; ++d) VtV[(size_t)i * kD + d] = ld(blob_vv_off(bd, es, d, i));
  if (UK) for (int t = 0; t < len; ++t) for (int i = 0; i < rk; ++i) UK[(size_t)t * rk + i] = ld(blob_uk_off(bd, es, t, i));
  if (UV) for (int t = 0; t < len; ++t) for (int i = 0; i < rv; ++i) UV[(size_t)t * rv + i] = ld(blob_uv_off(bd, es, t, i));
  if (pad_zero) {
    bool ok = true;
    for (int i = rk; i < bd.rkp; ++i) ok = ok && bsk[i] == 0.f;
    for (int i = rv; i < bd.rvp; ++i) ok = ok && bsv[i] == 0.f;
    for (int i = 0; i < bd.rkp && ok; ++i) for (int d = 0; d < kD; ++d) if (i >= rk && ld(blob_vtk_off(bd, es, i, d)) != 0.f) ok = false;
    for (int i = 0; i < bd.rvp && ok; ++i) for (int d = 0; d < kD; ++d) if (i >= rv && ld(blob_vv_off(bd, es, d, i)) != 0.f) ok = false;
    for (int t = 0; t < bd.lenp && ok; ++t) {
      for (int i = 0; i < bd.rkp; ++i) if ((t >= len || i >= rk) && ld(blob_uk_off(bd, es, t, i)) != 0.f) ok = false;
      for (int i = 0; i < bd.rvp; ++i) if ((t >= len || i >= rv) && ld(blob_uv_off(bd, es, t, i)) != 0.f) ok = false;
    }
    *pad_zero = ok ? 1 : 0;
  }
  return SEKV_OK;
}

sekv_status sekv_get_schedule(const sekv_handle* h, int32_t* stage1_ctas, int32_t* parts_per_head) {
  if (!h) return SEKV_INVALID_ARG;
  if (stage1_ctas) *stage1_ctas = h->n_chunks;
  if (parts_per_head) *parts_per_head = h->parts_per_head;
  return SEKV_OK;
}

}  // extern "C"

