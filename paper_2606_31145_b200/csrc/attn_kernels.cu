// a5-a7, generic kernels (any storage dtype, plain fp32 ALU math), one kernel per step.  Used for fp32
// storage (config 0), when cfg.impl = 1, and when a factor blob is too large for the fused kernel's
// shared-memory staging; the bf16 hot path is the fused layer kernel in fused_kernels.cu, checked against
// the same oracle.
//
// Softmax bookkeeping is in the base-2 domain: z = logit * log2(e); a partial is
// (m2 = max z, l = sum 2^(z - m2), o[128] = sum 2^(z - m2) v), merged by the combine kernel
// ("outputs merged across both stages", reading #18).
#include <algorithm>

#include "sekv_internal.cuh"

namespace sekv {


// ---------------------------------------------------------------------------------------------
// a5: stage 1 -- pool tokens (logit = q.K/sqrt(d)) and unexpanded coarse entries
// (logit = q.k_bar/sqrt(d) + ln|S|, value v_bar).
// One CTA (4 warps) per schedule chunk; a warp owns every 4th entry row; a lane owns 4 dims.
// ---------------------------------------------------------------------------------------------
constexpr int kS1Threads = 128;

template <typename ST, int G>
__global__ void __launch_bounds__(kS1Threads)
stage1_kernel(CsrView cv, LayerView lv, const Chunk* __restrict__ chunks, const ST* __restrict__ q, int Hq, int Hkv,
              size_t ent_head_stride, int mask_words, float* __restrict__ partials) {
  __shared__ float sh_m[4][G], sh_l[4][G];
  __shared__ float sh_o[4][G][kD];
  const Chunk ck = chunks[blockIdx.x];
  const int b = ck.bg / Hkv, g = ck.bg % Hkv;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int A = cv.seq_pool_cnt[b];
  const int row0 = cv.seq_row_off[b];
  const int span0 = cv.seq_span_off[b];
  const ST* K = (const ST*)lv.ent_k + (size_t)g * ent_head_stride + (size_t)row0 * kD;
  const ST* V = (const ST*)lv.ent_v + (size_t)g * ent_head_stride + (size_t)row0 * kD;
  const uint32_t* mask = lv.zoom_mask + (size_t)ck.bg * mask_words;
  const float scale2 = rsqrtf((float)kD) * kLog2e;
  float qr[G][4];
#pragma unroll
  for (int h = 0; h < G; ++h) ld4(q + ((size_t)b * Hq + (size_t)g * G + h) * kD + lane * 4, qr[h]);
  float m2[G], l[G], acc[G][4];
#pragma unroll
  for (int h = 0; h < G; ++h) { m2[h] = -INFINITY; l[h] = 0.f; acc[h][0] = acc[h][1] = acc[h][2] = acc[h][3] = 0.f; }
  for (int r = ck.row_begin + warp; r < ck.row_end; r += 4) {
    float bias2 = 0.f;
    if (r >= A) {
      const int s = r - A;
      if (mask[s >> 5] & (1u << (s & 31))) continue;        // expanded: replaced by its tokens (L121)
      bias2 = cv.ln_len[span0 + s] * kLog2e;
    }
    float k4[4], v4[4];
    ld4(K + (size_t)r * kD + lane * 4, k4);
    ld4(V + (size_t)r * kD + lane * 4, v4);
    float z[G];
#pragma unroll
    for (int h = 0; h < G; ++h) {
      float d = k4[0] * qr[h][0];
      d = fmaf(k4[1], qr[h][1], d); d = fmaf(k4[2], qr[h][2], d); d = fmaf(k4[3], qr[h][3], d);
      z[h] = fmaf(warp_sum(d), scale2, bias2);
    }
#pragma unroll
    for (int h = 0; h < G; ++h) {
      const float mn = fmaxf(m2[h], z[h]);
      const float corr = exp2f(m2[h] - mn);      // m2 = -inf on the first row: exp2(-inf) = 0
      const float p = exp2f(z[h] - mn);
      l[h] = fmaf(l[h], corr, p);
#pragma unroll
      for (int e = 0; e < 4; ++e) acc[h][e] = fmaf(acc[h][e], corr, p * v4[e]);
      m2[h] = mn;
    }
  }
  // merge the 4 warps
#pragma unroll
  for (int h = 0; h < G; ++h) {
    if (lane == 0) { sh_m[warp][h] = m2[h]; sh_l[warp][h] = l[h]; }
#pragma unroll
    for (int e = 0; e < 4; ++e) sh_o[warp][h][lane * 4 + e] = acc[h][e];
  }
  __syncthreads();
  const int d = threadIdx.x;   // 128 threads = 128 dims
  float* out = partials + (size_t)blockIdx.x * G * kPartStride;
#pragma unroll
  for (int h = 0; h < G; ++h) {
    float mm = fmaxf(fmaxf(sh_m[0][h], sh_m[1][h]), fmaxf(sh_m[2][h], sh_m[3][h]));
    float ls = 0.f, os = 0.f;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const float c = (sh_m[w][h] == -INFINITY) ? 0.f : exp2f(sh_m[w][h] - mm);
      ls = fmaf(sh_l[w][h], c, ls);
      os = fmaf(sh_o[w][h][d], c, os);
    }
    if (d == 0) { out[h * kPartStride] = mm; out[h * kPartStride + 1] = ls; }
    out[h * kPartStride + 4 + d] = os;
  }
}

template <typename ST>
static cudaError_t launch_stage1_t(sekv_handle* h, int layer, const void* q, cudaStream_t s) {
  const sekv_config& c = h->cfg;
  if (h->n_chunks == 0) return cudaSuccess;
  CsrView cv = csr_view(h);
  LayerView lv = layer_view(h, layer);
  const Chunk* chunks = (const Chunk*)ws(h, h->F.off_chunks);
  float* partials = (float*)ws(h, h->F.off_partials1);
  const size_t ehs = (size_t)h->lay.rows_cap * kD;
#define SEKV_S1(GG)                                                                                          \
  case GG:                                                                                                   \
    stage1_kernel<ST, GG><<<h->n_chunks, kS1Threads, 0, s>>>(cv, lv, chunks, (const ST*)q, c.n_q_heads,      \
                                                             c.n_kv_heads, ehs, h->mask_words, partials);    \
    break;
  switch (h->G) {
    SEKV_S1(1) SEKV_S1(2) SEKV_S1(3) SEKV_S1(4) SEKV_S1(5) SEKV_S1(6) SEKV_S1(7) SEKV_S1(8)
    default: return cudaErrorInvalidValue;
  }
#undef SEKV_S1
  h->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_stage1(sekv_handle* h, int layer, const void* q, cudaStream_t s) {
  if (h->cfg.dtype == SEKV_BF16) return launch_stage1_t<__nv_bfloat16>(h, layer, q, s);
  return launch_stage1_t<float>(h, layer, q, s);
}

// ---------------------------------------------------------------------------------------------
// a6: stage 2 -- expanded spans through the factored form (BASELINE.json north_star):
//   c[h]      = sigma_K o (Vt_K q_h)              [r_K]
//   logit_t   = U_K[t] . c[h] / sqrt(d)           (= (U Sigma V^T q)_t, Eq. 8 never materialised)
//   y[h]      = sum_t p_t U_V[t]                  [r_V]
//   o[h]      = (sigma_V o y[h]) Vt_V             [128]
// One CTA per (group of kStage2SpansPerCta items, kv head, sequence); blobs are read from the device
// factor-cache slots chosen by the plan kernel.
// ---------------------------------------------------------------------------------------------
constexpr int kS2Threads = 128;

template <typename ST, int G>
__global__ void __launch_bounds__(kS2Threads)
stage2_kernel(CsrView cv, LayerView lv, const int32_t* __restrict__ count, const ST* __restrict__ q, int Hq,
              int k_cap, int ways, int spans_cap, int64_t slot_bytes, float* __restrict__ partials) {
  __shared__ float sh_q[G][kD];
  __shared__ float sh_c[G][SEKV_MAX_RANK];
  __shared__ float sh_y[G][SEKV_MAX_RANK];
  __shared__ float sh_z[G][SEKV_MAX_SPAN_LEN];
  __shared__ float sh_red[4][G];
  __shared__ float run_m[G], run_l[G];
  const int p = blockIdx.x, g = blockIdx.y, b = blockIdx.z, Hkv = gridDim.y, P2 = gridDim.x;
  const int bg = b * Hkv + g;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int cnt = min(count[bg], k_cap);
  const float scale2 = rsqrtf((float)kD) * kLog2e;
  for (int o = tid; o < G * kD; o += kS2Threads)
    sh_q[o / kD][o % kD] = StTraits<ST>::ld(q + ((size_t)b * Hq + (size_t)g * G) * kD + o);
  if (tid < G) { run_m[tid] = -INFINITY; run_l[tid] = 0.f; }
  float run_o[G];                       // thread tid owns output dim tid
#pragma unroll
  for (int h = 0; h < G; ++h) run_o[h] = 0.f;
  __syncthreads();
  for (int j = p * kStage2SpansPerCta; j < min(cnt, (p + 1) * kStage2SpansPerCta); ++j) {
    const int id = lv.item_span[(size_t)bg * k_cap + j];
    if (id < 0) continue;                                                // dropped duplicate / invalid id
    const int way = (int)(lv.items[(size_t)bg * k_cap + j] & 0x7FFFFFFFu);
    const int gs = cv.seq_span_off[b] + id;
    const int rr = lv.dir_rank[(size_t)g * spans_cap + gs];
    const int len = cv.span_len[gs];
    const BlobDims bd = blob_dims((int)sizeof(ST), len, rr & 0xff, (rr >> 8) & 0xff);
    const uint8_t* blob = lv.slots + ((size_t)bg * ways + way) * slot_bytes;
    const float* sK = (const float*)(blob + bd.off_sk);
    const float* sV = (const float*)(blob + bd.off_sv);
    const int es = (int)sizeof(ST);
    // c[h][i]
    for (int o = tid; o < G * bd.rkp; o += kS2Threads) {
      const int h = o / bd.rkp, i = o % bd.rkp;
      float a = 0.f;
      for (int d = 0; d < kD; d += 4) {
        float v4[4];
        ld4((const ST*)(blob + blob_vtk_off(bd, es, i, d)), v4);
        a = fmaf(v4[0], sh_q[h][d], a); a = fmaf(v4[1], sh_q[h][d + 1], a);
        a = fmaf(v4[2], sh_q[h][d + 2], a); a = fmaf(v4[3], sh_q[h][d + 3], a);
      }
      sh_c[h][i] = a * sK[i] * scale2;
    }
    __syncthreads();
    // logits (base 2) and the span's max
    float mx[G];
#pragma unroll
    for (int h = 0; h < G; ++h) mx[h] = -INFINITY;
    for (int t = tid; t < len; t += kS2Threads) {
      float z[G];
#pragma unroll
      for (int h = 0; h < G; ++h) z[h] = 0.f;
      for (int i = 0; i < bd.rkp; i += 4) {
        float u4[4];
        ld4((const ST*)(blob + blob_uk_off(bd, es, t, i)), u4);
#pragma unroll
        for (int h = 0; h < G; ++h) {
          z[h] = fmaf(u4[0], sh_c[h][i], z[h]); z[h] = fmaf(u4[1], sh_c[h][i + 1], z[h]);
          z[h] = fmaf(u4[2], sh_c[h][i + 2], z[h]); z[h] = fmaf(u4[3], sh_c[h][i + 3], z[h]);
        }
      }
#pragma unroll
      for (int h = 0; h < G; ++h) { sh_z[h][t] = z[h]; mx[h] = fmaxf(mx[h], z[h]); }
    }
#pragma unroll
    for (int h = 0; h < G; ++h) { const float w = warp_max(mx[h]); if (lane == 0) sh_red[warp][h] = w; }
    __syncthreads();
    float mnew[G], corr[G];
#pragma unroll
    for (int h = 0; h < G; ++h) {
      const float ms = fmaxf(fmaxf(sh_red[0][h], sh_red[1][h]), fmaxf(sh_red[2][h], sh_red[3][h]));
      mnew[h] = fmaxf(run_m[h], ms);
      corr[h] = exp2f(run_m[h] - mnew[h]);
    }
    __syncthreads();                     // everyone has read run_m / sh_red
    // p_t = 2^(z - m), partial sums
    float ls[G];
#pragma unroll
    for (int h = 0; h < G; ++h) ls[h] = 0.f;
    for (int t = tid; t < bd.lenp; t += kS2Threads) {
#pragma unroll
      for (int h = 0; h < G; ++h) {
        const float pz = t < len ? exp2f(sh_z[h][t] - mnew[h]) : 0.f;
        sh_z[h][t] = pz;
        ls[h] += pz;
      }
    }
#pragma unroll
    for (int h = 0; h < G; ++h) { const float w = warp_sum(ls[h]); if (lane == 0) sh_red[warp][h] = w; }
    __syncthreads();
    if (tid < G) {
      run_l[tid] = run_l[tid] * corr[tid] + sh_red[0][tid] + sh_red[1][tid] + sh_red[2][tid] + sh_red[3][tid];
      run_m[tid] = mnew[tid];
    }
    // y[h][i] = sigma_V[i] * sum_t p[h][t] UVt[i][t]
    for (int o = tid; o < G * bd.rvp; o += kS2Threads) {
      const int h = o / bd.rvp, i = o % bd.rvp;
      float a = 0.f;
      for (int t = 0; t < bd.lenp; ++t)
        a = fmaf(StTraits<ST>::ld((const ST*)(blob + blob_uv_off(bd, es, t, i))), sh_z[h][t], a);
      sh_y[h][i] = a * sV[i];
    }
    __syncthreads();
    // o[h][d] += y[h] . VV[d]
    {
      float add[G];
#pragma unroll
      for (int h = 0; h < G; ++h) add[h] = 0.f;
      for (int i = 0; i < bd.rvp; ++i) {
        const float v = StTraits<ST>::ld((const ST*)(blob + blob_vv_off(bd, es, tid, i)));   // V_V[d = tid][i]
#pragma unroll
        for (int h = 0; h < G; ++h) add[h] = fmaf(v, sh_y[h][i], add[h]);
      }
#pragma unroll
      for (int h = 0; h < G; ++h) run_o[h] = fmaf(run_o[h], corr[h], add[h]);
    }
    __syncthreads();
  }
  float* out = partials + ((size_t)bg * P2 + p) * G * kPartStride;
#pragma unroll
  for (int h = 0; h < G; ++h) {
    if (tid == 0) { out[h * kPartStride] = run_m[h]; out[h * kPartStride + 1] = run_l[h]; }
    out[h * kPartStride + 4 + tid] = run_o[h];
  }
}

template <typename ST>
static cudaError_t launch_stage2_t(sekv_handle* h, int layer, const void* q, const int32_t* count, cudaStream_t s) {
  const sekv_config& c = h->cfg;
  CsrView cv = csr_view(h);
  LayerView lv = layer_view(h, layer);
  float* partials = (float*)ws(h, h->F.off_partials2);
  dim3 grid(h->P2, c.n_kv_heads, h->n_seqs);
#define SEKV_S2(GG)                                                                                              \
  case GG:                                                                                                       \
    stage2_kernel<ST, GG><<<grid, kS2Threads, 0, s>>>(cv, lv, count, (const ST*)q, c.n_q_heads, c.k_cap,         \
                                                      c.cache_ways, (int)h->lay.spans_cap, h->lay.slot_bytes,    \
                                                      partials);                                                 \
    break;
  switch (h->G) {
    SEKV_S2(1) SEKV_S2(2) SEKV_S2(3) SEKV_S2(4) SEKV_S2(5) SEKV_S2(6) SEKV_S2(7) SEKV_S2(8)
    default: return cudaErrorInvalidValue;
  }
#undef SEKV_S2
  h->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_stage2(sekv_handle* h, int layer, const void* q, const int32_t* count, cudaStream_t s) {
  if (h->cfg.k_cap <= 0) return cudaSuccess;
  if (h->cfg.dtype == SEKV_BF16) return launch_stage2_t<__nv_bfloat16>(h, layer, q, count, s);
  return launch_stage2_t<float>(h, layer, q, count, s);
}

// ---------------------------------------------------------------------------------------------
// a7: combine -- log-sum-exp merge of a head's partials (stage-1 chunks of its (sequence, kv head)
// and the stage-2 groups), normalise, write out and the natural-log lse.  Also advances the layer's
// step stamp for the cache LRU.
// ---------------------------------------------------------------------------------------------
template <typename OT>
__global__ void __launch_bounds__(kD)
combine_kernel(const int32_t* __restrict__ bg_chunk, const float* __restrict__ part1, const float* __restrict__ part2,
               int G, int P2, int use_p2, OT* __restrict__ out, float* __restrict__ lse, uint32_t* __restrict__ layer_step) {
  const int h = blockIdx.x, b = blockIdx.y, Hq = gridDim.x;
  const int Hkv = Hq / G, g = h / G, hl = h % G, bg = b * Hkv + g;
  const int d = threadIdx.x;
  const int c0 = bg_chunk[bg], c1 = bg_chunk[bg + 1];
  const int n2 = use_p2 ? P2 : 0;
  float mm = -INFINITY;
  for (int c = c0; c < c1; ++c) mm = fmaxf(mm, part1[((size_t)c * G + hl) * kPartStride]);
  for (int p = 0; p < n2; ++p) mm = fmaxf(mm, part2[(((size_t)bg * P2 + p) * G + hl) * kPartStride]);
  float L = 0.f, o = 0.f;
  if (mm != -INFINITY) {
    for (int c = c0; c < c1; ++c) {
      const float* pp = part1 + ((size_t)c * G + hl) * kPartStride;
      const float w = pp[0] == -INFINITY ? 0.f : exp2f(pp[0] - mm);
      L = fmaf(pp[1], w, L);
      o = fmaf(pp[4 + d], w, o);
    }
    for (int p = 0; p < n2; ++p) {
      const float* pp = part2 + (((size_t)bg * P2 + p) * G + hl) * kPartStride;
      const float w = pp[0] == -INFINITY ? 0.f : exp2f(pp[0] - mm);
      L = fmaf(pp[1], w, L);
      o = fmaf(pp[4 + d], w, o);
    }
  }
  const float res = L > 0.f ? o / L : 0.f;
  StTraits<OT>::st(out + ((size_t)b * Hq + h) * kD + d, res);
  if (lse && d == 0) lse[b * Hq + h] = L > 0.f ? (mm + log2f(L)) * kLn2 : -INFINITY;
  if (h == 0 && b == 0 && d == 0) *layer_step += 1u;
}

cudaError_t launch_combine(sekv_handle* h, int layer, void* out, float* lse, cudaStream_t s) {
  const sekv_config& c = h->cfg;
  LayerView lv = layer_view(h, layer);
  dim3 grid(c.n_q_heads, h->n_seqs);
  const int32_t* bgc = (const int32_t*)ws(h, h->F.off_bg_chunk);
  const float* p1 = (const float*)ws(h, h->F.off_partials1);
  const float* p2 = (const float*)ws(h, h->F.off_partials2);
  if (c.out_dtype == SEKV_BF16)
    combine_kernel<__nv_bfloat16><<<grid, kD, 0, s>>>(bgc, p1, p2, h->G, h->P2, c.k_cap > 0, (__nv_bfloat16*)out, lse, lv.layer_step);
  else
    combine_kernel<float><<<grid, kD, 0, s>>>(bgc, p1, p2, h->G, h->P2, c.k_cap > 0, (float*)out, lse, lv.layer_step);
  h->launches += 1;
  return cudaGetLastError();
}

}  // namespace sekv
