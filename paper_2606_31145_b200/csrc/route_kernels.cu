// a1-a3: query projection (Eq. 4), routing scores (Eq. 5), GQA reduce, threshold (Eq. 9) and top-k
// under the budget cap.  a4: device factor-cache residency plan and the
// pinned-host -> device-slot fetch.
#include <algorithm>

#include "sekv_internal.cuh"

namespace sekv {

// Monotone map float -> uint32 (larger float => larger key); -inf maps above 0, so key 0 is free to
// mean "not eligible / padding".
__device__ __forceinline__ uint32_t order_key(float x) {
  const uint32_t u = __float_as_uint(x);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

constexpr int kRouteThreads = 256;

// One CTA per (kv head, sequence).
//   q'[h] = W[h] q[h]                                   (Eq. 4)
//   x[h][s] = q'[h] . K_bar[h][s] / sqrt(d') + ln|S_s|  (Eq. 5, pre-sigmoid logit; alpha = sig(x))
//   X[s] = max_h x[h][s]; eligible iff no tau or alpha[h][s] > tau[h] for some h   (Eq. 9, reading #10)
//   ids = the min(k, #eligible) eligible spans of largest X, ties to the lower id    (L123)
// Selection: 64-bit keys (order(X) << 32 | ~s) sorted descending by a bitonic network in shared
// memory; intra-warp stages use shuffles.
template <typename ST>
__global__ void __launch_bounds__(kRouteThreads)
route_topk_kernel(CsrView cv, const ST* __restrict__ q, const ST* __restrict__ W, const ST* __restrict__ route,
                  size_t route_head_stride, const float* __restrict__ tau, int k, int k_cap, int Hq, int G, int dp,
                  int sort_n, int m_tot_stride, float* __restrict__ logits_out, float* __restrict__ alpha_out,
                  int32_t* __restrict__ ids, int32_t* __restrict__ count) {
  extern __shared__ unsigned long long keys[];            // [sort_n]
  __shared__ float sh_q[SEKV_MAX_GROUP * kD];
  __shared__ float sh_qp[SEKV_MAX_GROUP * SEKV_MAX_ROUTE_DIM];
  __shared__ int sh_elig;
  const int g = blockIdx.x, b = blockIdx.y, Hkv = gridDim.x, tid = threadIdx.x;
  const int span0 = cv.seq_span_off[b];
  const int m = cv.seq_span_off[b + 1] - span0;
  if (tid == 0) sh_elig = 0;
  for (int o = tid; o < G * kD; o += kRouteThreads)
    sh_q[o] = StTraits<ST>::ld(q + ((size_t)b * Hq + (size_t)g * G) * kD + o);
  __syncthreads();
  // Eq. 4: one thread per (head, j)
  for (int o = tid; o < G * dp; o += kRouteThreads) {
    const int hl = o / dp, j = o % dp;
    const ST* wr = W + ((size_t)(g * G + hl) * dp + j) * kD;
    float acc = 0.f;
    for (int d = 0; d < kD; d += 4) {
      float w4[4];
      ld4(wr + d, w4);
      acc = fmaf(w4[0], sh_q[hl * kD + d], acc); acc = fmaf(w4[1], sh_q[hl * kD + d + 1], acc);
      acc = fmaf(w4[2], sh_q[hl * kD + d + 2], acc); acc = fmaf(w4[3], sh_q[hl * kD + d + 3], acc);
    }
    sh_qp[o] = acc;
  }
  __syncthreads();
  const float inv_sqrt_dp = rsqrtf((float)dp);
  int my_elig = 0;
  for (int s = tid; s < sort_n; s += kRouteThreads) {
    unsigned long long key = 0ull;
    if (s < m) {
      const float lnl = cv.ln_len[span0 + s];
      float X = -INFINITY;
      bool elig = (tau == nullptr);
      for (int hl = 0; hl < G; ++hl) {
        const int h = g * G + hl;
        const ST* kr = route + (size_t)h * route_head_stride + (size_t)(span0 + s) * dp;
        float acc = 0.f;
        for (int j = 0; j < dp; j += 4) {
          float k4[4];
          ld4(kr + j, k4);
          acc = fmaf(k4[0], sh_qp[hl * dp + j], acc); acc = fmaf(k4[1], sh_qp[hl * dp + j + 1], acc);
          acc = fmaf(k4[2], sh_qp[hl * dp + j + 2], acc); acc = fmaf(k4[3], sh_qp[hl * dp + j + 3], acc);
        }
        const float x = fmaf(acc, inv_sqrt_dp, lnl);
        const float a = 1.f / (1.f + __expf(-x));
        if (logits_out) logits_out[(size_t)h * m_tot_stride + span0 + s] = x;
        if (alpha_out) alpha_out[(size_t)h * m_tot_stride + span0 + s] = a;
        if (tau != nullptr && a > tau[h]) elig = true;
        X = fmaxf(X, x);
      }
      if (elig) { key = ((unsigned long long)order_key(X) << 32) | (unsigned long long)(0xFFFFFFFFu - (uint32_t)s); ++my_elig; }
    }
    keys[s] = key;
  }
  if (my_elig) atomicAdd(&sh_elig, my_elig);
  __syncthreads();
  // bitonic sort, descending
  for (int size = 2; size <= sort_n; size <<= 1) {
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int i = tid; i < (sort_n >> 1); i += kRouteThreads) {
        const int lo = ((i & ~(stride - 1)) << 1) | (i & (stride - 1));
        const int hi = lo | stride;
        const bool desc = ((lo & size) == 0);
        const unsigned long long a = keys[lo], c = keys[hi];
        if ((a < c) == desc) { keys[lo] = c; keys[hi] = a; }
      }
      __syncthreads();
    }
  }
  const int n_elig = sh_elig;
  int cnt = k < 0 ? n_elig : min(k, n_elig);
  cnt = min(cnt, k_cap);
  int32_t* my_ids = ids + ((size_t)b * Hkv + g) * max(k_cap, 1);
  for (int j = tid; j < k_cap; j += kRouteThreads)
    my_ids[j] = j < cnt ? (int32_t)(0xFFFFFFFFu - (uint32_t)(keys[j] & 0xFFFFFFFFull)) : -1;
  if (tid == 0) count[b * Hkv + g] = cnt;
}

cudaError_t launch_route(sekv_handle* h, int layer, const void* q, const float* tau, int k, float* logits,
                         float* alpha, int32_t* ids, int32_t* count, cudaStream_t s) {
  const sekv_config& c = h->cfg;
  CsrView cv = csr_view(h);
  LayerView lv = layer_view(h, layer);
  dim3 grid(c.n_kv_heads, h->n_seqs);
  const size_t smem = (size_t)h->sort_n * 8;
  const size_t rhs = (size_t)h->lay.spans_cap * c.route_dim;
  if (c.dtype == SEKV_BF16) {
    if (smem > 48 * 1024) cudaFuncSetAttribute(route_topk_kernel<__nv_bfloat16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    route_topk_kernel<__nv_bfloat16><<<grid, kRouteThreads, smem, s>>>(
        cv, (const __nv_bfloat16*)q, (const __nv_bfloat16*)lv.W, (const __nv_bfloat16*)lv.route, rhs, tau, k, c.k_cap,
        c.n_q_heads, h->G, c.route_dim, h->sort_n, h->m_tot, logits, alpha, ids, count);
  } else {
    if (smem > 48 * 1024) cudaFuncSetAttribute(route_topk_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    route_topk_kernel<float><<<grid, kRouteThreads, smem, s>>>(
        cv, (const float*)q, (const float*)lv.W, (const float*)lv.route, rhs, tau, k, c.k_cap, c.n_q_heads, h->G,
        c.route_dim, h->sort_n, h->m_tot, logits, alpha, ids, count);
  }
  h->launches += 1;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// a4: residency plan.  One warp per (kv head, sequence).  The device factor cache of a (layer,
// sequence, kv head) is `ways` slots with a tag (span id) and a stamp (step of last use); spans in
// this step's zoom set that are resident are hits, the others take the least-recently-used slots
// not needed by this step.  Also: zoom bit-mask for stage 1 (an expanded span's coarse entry is
// replaced by its tokens), de-duplication of caller-supplied ids, statistics.
// ---------------------------------------------------------------------------------------------
constexpr int kPlanThreads = 32;

__global__ void __launch_bounds__(kPlanThreads)
plan_kernel(CsrView cv, LayerView lv, const int32_t* __restrict__ ids, const int32_t* __restrict__ count, int k_cap,
            int ways, int mask_words, int spans_cap, int esize, unsigned long long* __restrict__ stats) {
  extern __shared__ int sh[];          // tags[ways], stamps[ways], victim[ways]
  int* sh_tag = sh;
  uint32_t* sh_stamp = (uint32_t*)(sh + ways);
  int* sh_victim = sh + 2 * ways;
  const int g = blockIdx.x, b = blockIdx.y, Hkv = gridDim.x, lane = threadIdx.x;
  const int bg = b * Hkv + g;
  const int span0 = cv.seq_span_off[b];
  const int m = cv.seq_span_off[b + 1] - span0;
  const uint32_t cur = *lv.layer_step + 1u;
  int32_t* tags = lv.tags + (size_t)bg * ways;
  uint32_t* stamps = lv.stamps + (size_t)bg * ways;
  uint32_t* mask = lv.zoom_mask + (size_t)bg * mask_words;
  uint32_t* items = lv.items + (size_t)bg * max(k_cap, 1);
  int32_t* item_span = lv.item_span + (size_t)bg * max(k_cap, 1);
  const int32_t* my_ids = ids ? ids + (size_t)bg * max(k_cap, 1) : nullptr;
  int cnt = (count && ids) ? min(count[bg], k_cap) : 0;
  if (cnt < 0) cnt = 0;
  for (int w = lane; w < mask_words; w += 32) mask[w] = 0u;
  for (int w = lane; w < ways; w += 32) { sh_tag[w] = tags[w]; sh_stamp[w] = stamps[w]; }
  __syncwarp();
  unsigned long long n_hit = 0, n_miss = 0, bytes_algo = 0, bytes_h2d = 0;
  // pass 1: validate / de-duplicate, set mask bits, look up residency
  for (int j0 = 0; j0 < cnt; j0 += 32) {
    const int j = j0 + lane;
    int id = (j < cnt) ? my_ids[j] : -1;
    if (id < 0 || id >= m) id = -1;
    // de-duplicate: the first occurrence wins (lanes in order, then earlier chunks via the mask)
    for (int l = 0; l < 32; ++l) {            // serialise lanes so that test-and-set is ordered
      if (l == lane && id >= 0) {
        const uint32_t bit = 1u << (id & 31);
        if (mask[id >> 5] & bit) id = -1; else mask[id >> 5] |= bit;
      }
      __syncwarp();
    }
    int way = -1;
    if (id >= 0) {
      for (int w = 0; w < ways; ++w) if (sh_tag[w] == id) { way = w; break; }
    }
    if (j < cnt) { item_span[j] = id; items[j] = (way >= 0) ? (uint32_t)way : 0xFFFFFFFFu; }
    __syncwarp();
    if (way >= 0) { sh_stamp[way] = cur; ++n_hit; }
    __syncwarp();
    if (id >= 0) {
      const int rr = lv.dir_rank[(size_t)g * spans_cap + span0 + id];
      const int rk = rr & 0xff, rv = (rr >> 8) & 0xff;
      const int len = cv.span_len[span0 + id];
      bytes_algo += (unsigned long long)(rk + rv) * (len + kD) * esize + 4ull * (rk + rv);
      if (way < 0) { ++n_miss; bytes_h2d += blob_dims(esize, len, rk, rv).bytes; }
    }
  }
  __syncwarp();
  // victims: ways not used by this step, oldest stamp first (ties to the lower way)
  for (int w = lane; w < ways; w += 32) {
    int rank = -1;
    if (sh_stamp[w] != cur) {
      rank = 0;
      const uint32_t mine = sh_stamp[w];
      for (int v = 0; v < ways; ++v) {
        const uint32_t o = sh_stamp[v];
        rank += (o != cur) && (o < mine || (o == mine && v < w));
      }
    }
    if (rank >= 0) sh_victim[rank] = w;
  }
  __syncwarp();
  // pass 2: misses take victims in order
  int miss_base = 0;
  for (int j0 = 0; j0 < cnt; j0 += 32) {
    const int j = j0 + lane;
    const bool miss = (j < cnt) && item_span[j] >= 0 && items[j] == 0xFFFFFFFFu;
    const unsigned bal = __ballot_sync(0xffffffffu, miss);
    if (miss) {
      const int way = sh_victim[miss_base + __popc(bal & ((1u << lane) - 1u))];
      sh_tag[way] = item_span[j];
      sh_stamp[way] = cur;
      items[j] = (uint32_t)way | 0x80000000u;
    }
    miss_base += __popc(bal);
    __syncwarp();
  }
  for (int w = lane; w < ways; w += 32) { tags[w] = sh_tag[w]; stamps[w] = sh_stamp[w]; }
  // statistics
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    n_hit += __shfl_xor_sync(0xffffffffu, n_hit, o);
    n_miss += __shfl_xor_sync(0xffffffffu, n_miss, o);
    bytes_algo += __shfl_xor_sync(0xffffffffu, bytes_algo, o);
    bytes_h2d += __shfl_xor_sync(0xffffffffu, bytes_h2d, o);
  }
  if (lane == 0) {
    if (n_hit) atomicAdd(&stats[ST_HITS], n_hit);
    if (n_miss) atomicAdd(&stats[ST_MISSES], n_miss);
    if (n_hit + n_miss) { atomicAdd(&stats[ST_ZOOMED], n_hit + n_miss); atomicAdd(&stats[ST_SKIPPED], n_hit + n_miss); }
    if (bytes_algo) atomicAdd(&stats[ST_FACTOR_ALGO], bytes_algo);
    if (bytes_h2d) atomicAdd(&stats[ST_H2D], bytes_h2d);
    if (bg == 0) atomicAdd(&stats[ST_LAYER_STEPS], 1ull);
  }
}

cudaError_t launch_plan(sekv_handle* h, int layer, const int32_t* ids, const int32_t* count, cudaStream_t s) {
  const sekv_config& c = h->cfg;
  dim3 grid(c.n_kv_heads, h->n_seqs);
  const size_t smem = (size_t)c.cache_ways * 12;
  if (smem > 48 * 1024) cudaFuncSetAttribute(plan_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  plan_kernel<<<grid, kPlanThreads, smem, s>>>(csr_view(h), layer_view(h, layer), ids, count, c.k_cap, c.cache_ways,
                                               h->mask_words, (int)h->lay.spans_cap, h->esize,
                                               (unsigned long long*)ws(h, h->F.off_stats));
  h->launches += 1;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// a4: fetch.  Side stream.  One CTA per (item, kv head, sequence); items that hit the cache exit at
// once.  The blob is read straight from the pinned host arena through its device mapping (PCIe reads
// issued by the SMs, 16 bytes per thread, 4 in flight) and written to the cache slot.
// ---------------------------------------------------------------------------------------------
constexpr int kFetchThreads = 256;

__global__ void __launch_bounds__(kFetchThreads)
fetch_kernel(CsrView cv, LayerView lv, const int32_t* __restrict__ count, int k_cap, int ways, int spans_cap,
             int esize, int64_t slot_bytes, const uint8_t* __restrict__ host_arena) {
  const int j = blockIdx.x, g = blockIdx.y, b = blockIdx.z, Hkv = gridDim.y;
  const int bg = b * Hkv + g;
  if (j >= min(count[bg], k_cap)) return;
  const uint32_t it = lv.items[(size_t)bg * k_cap + j];
  const int id = lv.item_span[(size_t)bg * k_cap + j];
  if (id < 0 || !(it & 0x80000000u)) return;
  const int way = (int)(it & 0x7FFFFFFFu);
  const int gs = cv.seq_span_off[b] + id;
  const int rr = lv.dir_rank[(size_t)g * spans_cap + gs];
  const BlobDims bd = blob_dims(esize, cv.span_len[gs], rr & 0xff, (rr >> 8) & 0xff);
  const int4* src = reinterpret_cast<const int4*>(host_arena + lv.dir_off[(size_t)g * spans_cap + gs]);
  int4* dst = reinterpret_cast<int4*>(lv.slots + ((size_t)bg * ways + way) * slot_bytes);
  const int n = (int)(bd.bytes / 16);
  int i = threadIdx.x;
  for (; i + 3 * kFetchThreads < n; i += 4 * kFetchThreads) {
    const int4 a = src[i], c = src[i + kFetchThreads], d = src[i + 2 * kFetchThreads], e = src[i + 3 * kFetchThreads];
    dst[i] = a; dst[i + kFetchThreads] = c; dst[i + 2 * kFetchThreads] = d; dst[i + 3 * kFetchThreads] = e;
  }
  for (; i < n; i += kFetchThreads) dst[i] = src[i];
}

cudaError_t launch_fetch(sekv_handle* h, int layer, const int32_t* count, cudaStream_t s) {
  const sekv_config& c = h->cfg;
  if (c.k_cap <= 0) return cudaSuccess;
  dim3 grid(c.k_cap, c.n_kv_heads, h->n_seqs);
  fetch_kernel<<<grid, kFetchThreads, 0, s>>>(csr_view(h), layer_view(h, layer), count, c.k_cap, c.cache_ways,
                                              (int)h->lay.spans_cap, h->esize, h->lay.slot_bytes, h->host_dev);
  h->launches += 1;
  return cudaGetLastError();
}

}  // namespace sekv
