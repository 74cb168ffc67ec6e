// Internal declarations shared by the translation units of libsekv (not part of the ABI).
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "sekv.h"

namespace sekv {

constexpr int kD = SEKV_HEAD_DIM;   // d_h
constexpr int kRankPad = 16;        // ranks padded to a multiple of this in a blob (one mma k-step)
constexpr int kLenPad = 16;         // |S| padded to a multiple of this in a blob
constexpr int kTile = 16;           // stage-1 schedules entry rows in tiles of 16
constexpr int kPartStride = kD + 4; // floats per partial: m2, l, pad, pad, o[128]
constexpr int kStage2SpansPerCta = 4;

__host__ __device__ inline int round_up(int x, int m) { return (x + m - 1) / m * m; }
__host__ __device__ inline size_t round_up_sz(size_t x, size_t m) { return (x + m - 1) / m * m; }

// ---- factor blob layout ------------------------------------------------
// Every operand is stored in the FRAGMENT ORDER of the warp-level mma.sync.m16n8k16 that consumes it in
// the fused layer kernel: a block of 32 lanes x 16 bytes (8 elements) per fragment load, lane = 4 gid + t4,
// so that each load is one 16-byte access per lane at consecutive addresses (coalesced from global memory,
// bank-conflict free from shared memory).  nks / nvs = ceil(rank_k / 16), ceil(rank_v / 16).
//   header : [sigma_K f32 16 nks][sigma_V f32 16 nvs]
//            [VtK : nks x (2 u x 4 jj) blocks]   B operand of c = Vt_K q   (rows = rank index, cols = d)
//            [VV  : nvs x 8 md blocks]           A operand of O^T = V_V (sigma_V o y)^T
//   chunks : ceil(|S| / 16) chunks of 16 tokens, each [U_K : nks blocks][U_V : nvs blocks]
//            U_K = B operand of S = c U_K^T, U_V = A operand of y^T = U_V^T P^T
// The header and any run of chunks are contiguous pieces (1-D bulk copies).  Element positions are given by
// the blob_*_off functions below; the pack kernel, the generic kernels and the export go through them.
struct BlobDims {
  int len, lenp, rk, rv, rkp, rvp, nks, nvs;
  size_t off_sk, off_sv, off_vtk, off_vv, off_chunks, chunk_bytes, bytes;
};
__host__ __device__ inline BlobDims blob_dims(int esize, int len, int rk, int rv) {
  BlobDims b;
  b.len = len; b.rk = rk; b.rv = rv;
  b.lenp = round_up(len, kLenPad);
  b.rkp = round_up(rk > 0 ? rk : 1, kRankPad);
  b.rvp = round_up(rv > 0 ? rv : 1, kRankPad);
  b.nks = b.rkp / 16; b.nvs = b.rvp / 16;
  size_t o = 0;
  b.off_sk = o;  o += (size_t)b.rkp * 4;
  b.off_sv = o;  o += (size_t)b.rvp * 4;
  b.off_vtk = o; o += (size_t)b.rkp * kD * esize;
  b.off_vv = o;  o += (size_t)kD * b.rvp * esize;
  b.off_chunks = o;
  b.chunk_bytes = (size_t)kLenPad * (b.rkp + b.rvp) * esize;
  o += (size_t)(b.lenp / kLenPad) * b.chunk_bytes;
  b.bytes = round_up_sz(o, 128);
  return b;
}
// byte offset of Vt_K[i][d] (i = rank index): block (ks, u, jj), lane (gid, t4), element e8 with
// i = 16 ks + 4 (gid >> 1) + 2 u + (gid & 1),  d = 32 jj + 8 t4 + e8
__host__ __device__ inline size_t blob_vtk_off(const BlobDims& b, int esize, int i, int d) {
  const int ks = i >> 4, il = i & 15;
  const int u = (il >> 1) & 1, gid = 2 * (il >> 2) + (il & 1);
  const int jj = d >> 5, t4 = (d & 31) >> 3, e8 = d & 7;
  return b.off_vtk + ((size_t)((((ks * 2 + u) * 4 + jj) * 32 + gid * 4 + t4) * 8 + e8)) * esize;
}
// byte offset of V_V[d][i] = Vt_V[i][d]: block (kv, md), lane (gid, t4), register a_{2 half + hi}, element e with
// d = 16 md + 8 hi + gid,  i = 16 kv + 8 half + 2 t4 + e
__host__ __device__ inline size_t blob_vv_off(const BlobDims& b, int esize, int d, int i) {
  const int kv = i >> 4, il = i & 15;
  const int half = il >> 3, t4 = (il & 7) >> 1, e = il & 1;
  const int md = d >> 4, hi = (d & 15) >> 3, gid = d & 7;
  return b.off_vv + ((size_t)(((kv * 8 + md) * 32 + gid * 4 + t4) * 8 + (half * 2 + hi) * 2 + e)) * esize;
}
// byte offset of U_K[t][i]: chunk t / 16, block ks, lane (gid, t4), n-tile nt, element e4 with
// t = 16 c + 8 nt + gid,  i = 16 ks + 4 t4 + e4
__host__ __device__ inline size_t blob_uk_off(const BlobDims& b, int esize, int t, int i) {
  const int tl = t & 15, nt = tl >> 3, gid = tl & 7;
  const int ks = i >> 4, t4 = (i & 15) >> 2, e4 = i & 3;
  return b.off_chunks + (size_t)(t >> 4) * b.chunk_bytes + ((size_t)((ks * 32 + gid * 4 + t4) * 8 + nt * 4 + e4)) * esize;
}
// byte offset of U_V[t][i]: chunk t / 16, block nks + mv, lane (gid, t4), register a_{2 half + hi}, element e with
// t = 16 c + 8 half + 2 t4 + e,  i = 16 mv + 8 hi + gid
__host__ __device__ inline size_t blob_uv_off(const BlobDims& b, int esize, int t, int i) {
  const int tl = t & 15, half = tl >> 3, t4 = (tl & 7) >> 1, e = tl & 1;
  const int mv = i >> 4, hi = (i & 15) >> 3, gid = i & 7;
  return b.off_chunks + (size_t)(t >> 4) * b.chunk_bytes +
         ((size_t)(((b.nks + mv) * 32 + gid * 4 + t4) * 8 + (half * 2 + hi) * 2 + e)) * esize;
}

// ---- device views ------------------------------------------------------------------------------
struct CsrView {
  const int64_t* seq_tok_off;
  const int32_t* seq_row_off;
  const int32_t* seq_span_off;
  const int32_t* seq_pool_cnt;
  const int32_t* span_len;
  const int64_t* span_tok_start;
  const float* ln_len;
  const int64_t* pool_tok;
};

struct LayerView {
  const void* ent_k;       // [H_kv][rows_cap][128]
  const void* ent_v;
  const void* route;       // [H][spans_cap][d']
  const void* W;           // [H][d'][128]
  const int64_t* dir_off;  // [H_kv][spans_cap]
  const int32_t* dir_rank;
  int32_t* tags;           // [B][H_kv][ways]
  uint32_t* stamps;
  uint8_t* slots;          // [B][H_kv][ways][slot_bytes]
  uint32_t* layer_step;    // [1]
  uint32_t* zoom_mask;     // [B][H_kv][mask_words]
  uint32_t* items;         // [B][H_kv][kc]  way | miss << 31, valid for j < count (kc = max(k_cap,1) + prefetch)
  int32_t* item_span;      // [B][H_kv][kc]  local span id (deduplicated; -1 = dropped)
};

struct Dims {
  int L, Hq, Hkv, G, dp, B, k_cap, ways, mask_words;
  int rows_cap, spans_cap;
  int esize;
  int64_t slot_bytes;
  int parts1_max, P2, parts_per_head;
};

struct Chunk {  // one stage-1 work item
  int32_t bg;         // b * H_kv + g
  int32_t row_begin;  // local entry row range within the sequence
  int32_t row_end;
  int32_t part;       // partial slot within the head
};

enum StatIdx { ST_LAYER_STEPS = 0, ST_ZOOMED, ST_HITS, ST_MISSES, ST_H2D, ST_FACTOR_ALGO, ST_SKIPPED, ST_PREFETCHED, ST_PF_BYTES, ST_COUNT = 10 };

// ---- fused layer kernel (fused_kernels.cu) -------------------------------------------------------
// Work items of the per-layer persistent kernel.  Every item is processed by ONE warp, claimed in queue order:
// POOL, COARSE (L119-121), ZOOM (Eq. 8), COMBINE (L61).  The chain a1-a4 of a group (q' = W q, routing scores,
// top-k, factor-cache plan) is not an item: a team of warps runs it at the start of the kernel (IT_SELECT is its
// trace record).
enum ItemKind { IT_PREFETCH = 1, IT_SELECT = 2, IT_POOL = 3, IT_ZOOM = 4, IT_COARSE = 5, IT_COMBINE = 6 };
enum FusedMode { FM_ROUTE = 1, FM_ATTN = 2 };   // FM_ATTN without FM_ROUTE: caller-supplied zoom set
struct __align__(16) Item {   // 48 bytes: three 16-byte loads
  int32_t kind;        // ItemKind
  int32_t bg;          // b * H_kv + g
  int32_t a, b;        // COMBINE: a = head within the group, b = POOL + COARSE partials; POOL / COARSE: entry-row
                       // range; ZOOM: a = descriptor index; PREFETCH: a = candidate index
  int32_t part;        // partial slot within the group (attention items)
  int32_t A;           // pool rows of the sequence
  int32_t row0;        // first entry row of the sequence
  int32_t span0;       // first span of the sequence
  int32_t pbase;       // first partial record of the group (records of kPartStride floats)
  int32_t np;          // partials per head of the group
  int32_t pad0, pad1;
};

struct __align__(16) ZDescG {   // what a ZOOM item needs to know about one expanded span (written by the plan)
  unsigned long long src;       // blob address: cache slot (hit) or device alias of the pinned-host store (miss)
  uint32_t bytes;
  uint32_t epoch0;              // the layer's step stamp: both halves carry it, ZOOM items poll until it matches
  uint32_t len_rr;              // |S| << 16 | rank_k | rank_v << 8
  uint32_t way_miss;            // way | j << 14 | way-pending << 29 | no-slot << 30 | miss << 31
  int32_t id;                   // local span id, -1 = dropped duplicate
  uint32_t epoch1;
};

struct FusedParams {
  CsrView cv;
  LayerView lv;
  const __nv_bfloat16* q;      // [B][H][128]
  const float* tau;            // [H] or null
  float* logits_out;           // [H][m_tot] or null
  float* alpha_out;
  int32_t* ids;                // [B][H_kv][k_cap]: written (FM_ROUTE) or read (caller-supplied zoom set)
  int32_t* count;              // [B][H_kv]
  void* out;                   // [B][H][128]
  float* lse;                  // [B][H] or null
  const Item* items;
  const int2* grp;             // [BG] first span and span count of the group's sequence
  float* partials;             // records [pbase + hl * np + part][kPartStride]
  ZDescG* zdesc;               // [BG][kc] of this layer
  int32_t* ctrs;               // [0] launch sequence number of the layer, then two counter sets (fused_kernels.cu)
  int32_t ctrs_set;            // ints per set
  int32_t* plan_counts;        // [BG][2] = n_zoom, n_cand
  LayerView pf_lv;             // the previous layer of the step: its prefetch candidates are copied by this launch
  const int32_t* pf_plan_counts;   // (null: nothing to copy)
  int32_t pf_early;                // pf_lv is the layer two launches back: its copies run before the dependency wait
  unsigned long long* stats;
  const uint8_t* host_arena;   // device alias of the pinned host factor store
  unsigned long long* trace;   // null, or 8 x u64 per item (sekv_set_trace)
  const uint8_t* next_W;       // W and routing table of the layer that runs next: prefetched into L2 by exiting warps
  const uint8_t* next_route;
  size_t next_W_bytes, next_route_head_bytes;
  size_t ent_head_stride, route_head_stride;
  int64_t slot_bytes, trace_cap;
  uint2* zmask2;               // [BG][mask_words] (zoom bits, step stamp) pairs of this layer
  uint2* zway;                 // [BG][kc] (it, step stamp) of the demand misses of this layer: their slot, published after the descriptor
  int32_t main_end;                              // number of work items of this launch
  int32_t mode, k, k_cap, prefetch, kc, BG;
  int32_t Hq, Hkv, dp, ways, mask_words, spans_cap, m_tot, out_bf16;
  int32_t region_bytes;                          // per-warp shared-memory region
  int32_t hoist;                                 // the chain's static part may run before the PDL wait
  int32_t team_warps, has_chain;                 // warps 0 .. team_warps-1 of CTA bg % grid run the chain of group bg
  int32_t route_spans, route_bufs;               // spans per routing block, staging buffers per team warp (1 or 2)
  int32_t sm_stage, stage_bytes;                 // staging buffers: dsm + sm_stage + warp * stage_bytes
  int32_t sm_keys, sm_cand, sm_ids, sm_wayof, sm_tags, sm_mask, sm_hist, sm_meta, sm_lnl, sm_qp;   // team tables (byte offsets)
};

// ---- storage-type helpers ------------------------------------------------------------------------
template <typename ST> struct StTraits;
template <> struct StTraits<float> {
  static __device__ __forceinline__ float ld(const float* p) { return *p; }
  static __device__ __forceinline__ void st(float* p, float v) { *p = v; }
};
template <> struct StTraits<__nv_bfloat16> {
  static __device__ __forceinline__ float ld(const __nv_bfloat16* p) { return __bfloat162float(*p); }
  static __device__ __forceinline__ void st(__nv_bfloat16* p, float v) { *p = __float2bfloat16_rn(v); }
};

// load 4 consecutive storage elements as floats (16-byte aligned for f32, 8-byte for bf16)
__device__ __forceinline__ void ld4(const float* p, float (&o)[4]) {
  float4 v = *reinterpret_cast<const float4*>(p);
  o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w;
}
__device__ __forceinline__ void ld4(const __nv_bfloat16* p, float (&o)[4]) {
  uint2 v = *reinterpret_cast<const uint2*>(p);
  o[0] = __uint_as_float(v.x << 16); o[1] = __uint_as_float(v.x & 0xffff0000u);
  o[2] = __uint_as_float(v.y << 16); o[3] = __uint_as_float(v.y & 0xffff0000u);
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// exp2 that maps (-inf) - (-inf) safely: callers guard m == -inf themselves
__device__ __forceinline__ float fast_exp2(float x) { return exp2f(x); }

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

}  // namespace sekv

// ---- host handle -----------------------------------------------------------------------------------
struct GraphEntry {
  const void* q; const float* tau; int32_t k; void* out; float* lse;
  cudaGraphExec_t exec;
  uint64_t nodes;
};

// Complete device-arena layout: the public tables (sekv_layout) plus workspace offsets.
struct FullLayout {
  sekv_layout lay;
  int64_t off_partials1, off_partials2, off_ws_ids, off_ws_count, off_stats, off_chunks, off_bg_chunk,
      off_zoom_mask, off_items, off_item_span, off_layer_step, off_seg_flag, off_seg_flag2, off_seg_len,
      off_seg_misc, off_q_stage, off_out_stage, off_lse_stage, off_err_flag, off_items_sched, off_bg_part,
      off_bg_route, off_ctrs, off_plan_counts, off_zdesc, off_zmask2, off_zway;
  int mask_words, max_chunks, max_items, ctrs_per_layer;
  size_t total;
};

struct sekv_handle {
  sekv_config cfg;
  int G, esize;
  uint8_t* dev; size_t dev_bytes;
  uint8_t* host; size_t host_bytes;
  uint8_t* host_dev;                 // device alias of the pinned host arena
  bool registered_host;
  sekv_layout lay;
  FullLayout F;
  int mask_words;
  cudaStream_t main, side;
  bool own_side;
  cudaEvent_t ev_fork, ev_join;
  // batch state
  int n_seqs; bool segmented;
  std::vector<int> m_b, A_b;
  std::vector<int64_t> tok_off;
  std::vector<int32_t> span_len_host;
  int m_tot, A_tot, max_m;
  std::vector<char> layer_built;
  size_t host_used;
  // schedule
  int n_chunks, parts1_max, P2, parts_per_head, sort_n;
  // fused layer kernel (bf16 path)
  bool use_fused, use_pdl;
  std::string fused_why;             // why the batch runs on the generic path (empty when use_fused)
  int n_items, pool_end, fused_grid, fused_item_rows;
  int num_sms;
  std::vector<GraphEntry> graphs;
  uint64_t launches;
  int pending_prefetch;              // layer whose speculative prefetch copies have not been carried out yet (-1: none)
  int pending_prefetch2;             // a second such layer (the one before it), or -1
  // per-kernel-class CUDA-event timing (sekv_set_profiling)
  bool profiling;
  void* trace_buf; int64_t trace_cap;
  struct ProfRec { int cls; cudaEvent_t a, b; };
  std::vector<ProfRec> prof;
  std::string err;
};

namespace sekv {

inline Dims make_dims(const sekv_handle* h) {
  Dims d;
  d.L = h->cfg.n_layers; d.Hq = h->cfg.n_q_heads; d.Hkv = h->cfg.n_kv_heads; d.G = h->G;
  d.dp = h->cfg.route_dim; d.B = h->n_seqs; d.k_cap = h->cfg.k_cap; d.ways = h->cfg.cache_ways;
  d.mask_words = h->mask_words;
  d.rows_cap = (int)h->lay.rows_cap; d.spans_cap = (int)h->lay.spans_cap; d.esize = h->esize;
  d.slot_bytes = h->lay.slot_bytes;
  d.parts1_max = h->parts1_max; d.P2 = h->P2; d.parts_per_head = h->parts_per_head;
  return d;
}

CsrView csr_view(const sekv_handle* h);
LayerView layer_view(const sekv_handle* h, int layer);

// launchers (each returns the cudaError_t of the launch)
cudaError_t launch_segment(sekv_handle* h, const float* H, int n_seqs, const int64_t* tok_off_host,
                           int* m_out, int* a_out, std::string* why);
cudaError_t segment_scan(const float* H, int n_seqs, const int64_t* tok_off_dev, double alpha, int window, int l_min,
                         int max_span_len, uint8_t* flag, uint8_t* flag2, int32_t* len_at, double* thr,
                         int32_t* counts, int* err, cudaStream_t s);
cudaError_t launch_build_prefactored(sekv_handle* h, int layer, const float* H, const sekv_factors* f,
                                     const void* W);
cudaError_t launch_build_dense(sekv_handle* h, int layer, const float* H, const void* K, const void* V,
                               const void* W, int rank_cap, std::string* why);
cudaError_t launch_route(sekv_handle* h, int layer, const void* q, const float* tau, int k, float* logits,
                         float* alpha, int32_t* ids, int32_t* count, cudaStream_t s);
cudaError_t launch_plan(sekv_handle* h, int layer, const int32_t* ids, const int32_t* count, cudaStream_t s);
cudaError_t launch_fetch(sekv_handle* h, int layer, const int32_t* count, cudaStream_t s);
cudaError_t launch_stage1(sekv_handle* h, int layer, const void* q, cudaStream_t s);
cudaError_t launch_stage2(sekv_handle* h, int layer, const void* q, const int32_t* count, cudaStream_t s);
cudaError_t launch_combine(sekv_handle* h, int layer, void* out, float* lse, cudaStream_t s);
cudaError_t launch_fused(sekv_handle* h, int layer, int mode, const void* q, const float* tau, int k, float* logits,
                         float* alpha, int32_t* ids, int32_t* count, void* out, float* lse, cudaStream_t s);
bool fused_geometry(const sekv_handle* h, FusedParams* P, std::string* why);
cudaError_t launch_prefetch(sekv_handle* h, int layer, cudaStream_t s);
cudaError_t fused_occupancy(const sekv_handle* h, int* ctas_per_sm);
int fused_warps();

inline uint8_t* ws(const sekv_handle* h, int64_t off) { return h->dev + off; }

}  // namespace sekv
