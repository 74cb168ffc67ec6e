// The bf16 hot path: ONE persistent kernel per layer-step that runs a1-a7 (Eq. 4, 5, 9, L123,
// L119-121, Eq. 8) as work items pulled from a dependency-ordered queue:
//
//   ROUTE  (b, g, span chunk)   q' = W q, x = q'.K_bar/sqrt(d') + ln|S|, alpha = sig(x), X = max over the
//                               group, 64-bit keys -> global.  The LAST chunk of a (b, g) to finish sorts
//                               the keys (top-k, ties to the lower id), runs the residency plan of the
//                               device factor cache (LRU) and releases plan_flag[b, g].
//   POOL   (b, g, row range)    online-softmax partial over full-resolution tokens (no dependency).
//   ZOOM   (b, g, item range)   expanded spans through the factored form: the span's factor blob is moved
//                               by ONE 1-D bulk async copy (TMA engine) into shared memory -- from its cache
//                               slot on a hit, straight from the pinned-host store over PCIe on a demand
//                               miss (and then written to the slot) -- double-buffered across spans.
//   COARSE (b, g, row range)    partial over the unexpanded coarse entries (+ln|S|); needs the zoom mask.
//
// ZOOM and COARSE items wait on plan_flag[b, g]; the queue order (ROUTE, POOL..., ZOOM, COARSE) is a
// topological order and items are claimed in queue order, so a waiting CTA only ever waits on work that
// a running CTA has already claimed: no co-residency assumption, no deadlock.  The LAST attention item of
// a (b, g) to finish merges that group's partials by log-sum-exp and writes the output (a7).
//
// Tensor cores: G <= 8 query heads per kv head is far below a tcgen05 tile and the path is HBM-bound, so
// the heads are the (padded) 16 rows of warp-level mma.sync.m16n8k16 tiles; K/V rows stream from global
// memory straight into B fragments (every byte read once, coalesced 16-byte loads).
#include <algorithm>

#include "mma_common.cuh"

namespace sekv {

namespace {

constexpr int kFT = 128;        // threads per CTA
constexpr int kFW = kFT / 32;   // warps per CTA
constexpr int kCombineMaxParts = 512;

// Monotone map float -> uint32 (larger float => larger key); key 0 is free to mean "not eligible".
__device__ __forceinline__ uint32_t order_key(float x) {
  const uint32_t u = __float_as_uint(x);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

struct ZDesc { int32_t valid, miss, len, rr, way; uint32_t bytes; };

struct __align__(16) Shared {
  uint64_t bars[2];
  ZDesc desc[2];
  int32_t item, flag, scan[kFW + 1], misc[4];
  float ml[kFW * SEKV_MAX_GROUP * 2];
};

// ---------------------------------------------------------------------------------------------------
// a7: merge the warps' results of one CTA and store one partial (m2, l, o[128]) per head.
// ---------------------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ void cta_merge_store(float* sm_o, float* sm_ml, float* __restrict__ out) {
  __syncthreads();
  for (int o = threadIdx.x; o < G * kD; o += kFT) {
    const int h = o / kD, d = o % kD;
    float mm = -INFINITY;
#pragma unroll
    for (int w = 0; w < kFW; ++w) mm = fmaxf(mm, sm_ml[(w * G + h) * 2]);
    float ls = 0.f, os = 0.f;
#pragma unroll
    for (int w = 0; w < kFW; ++w) {
      const float mw = sm_ml[(w * G + h) * 2];
      const float c = (mw == -INFINITY) ? 0.f : exp2f(mw - mm);
      ls = fmaf(sm_ml[(w * G + h) * 2 + 1], c, ls);
      os = fmaf(sm_o[(w * G + h) * kD + d], c, os);
    }
    if (d == 0) { out[h * kPartStride] = mm; out[h * kPartStride + 1] = ls; }
    out[h * kPartStride + 4 + d] = os;
  }
}

__device__ __forceinline__ void load_q_frags(const __nv_bfloat16* __restrict__ q, int G, int gid, int t4,
                                             uint32_t (&qf)[4][4]) {
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (gid < G) v = *reinterpret_cast<const uint4*>(q + (size_t)gid * kD + (t4 + 4 * j) * 8);
    qf[j][0] = v.x; qf[j][1] = v.y; qf[j][2] = v.z; qf[j][3] = v.w;
  }
}

// ---------------------------------------------------------------------------------------------------
// a5: rows [row_begin, row_end) of the entry table of (b, g): pool tokens (logit = q.K/sqrt(d)) and
// unexpanded coarse entries (logit = q.k_bar/sqrt(d) + ln|S|, value v_bar).
//   QK^T : lane (gid = lane/4, t4 = lane%4) loads 16-byte chunk (t4 + 4j) of the K row of token gid; its
//          four words are the (b0,b1) pairs of two k-steps; Q is loaded the same way (the contraction
//          index may be permuted consistently on both operands).
//   P V  : computed transposed, O^T = V^T P^T (M = 16 dims, N = 8 heads, K = 16 tokens): the C fragment
//          of S IS the B fragment of P^T.  P (fp32) is split into bf16 hi + lo parts and multiplied
//          twice, so probabilities carry ~16 bits.
// ---------------------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ void rows_item(const FusedParams& P, int bg, int row_begin, int row_end, float* sm_o,
                                          float* sm_ml, float* __restrict__ partial_out) {
  const int b = bg / P.Hkv, g = bg % P.Hkv;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int gid = lane >> 2, t4 = lane & 3;
  const int A = P.cv.seq_pool_cnt[b];
  const int row0 = P.cv.seq_row_off[b];
  const int span0 = P.cv.seq_span_off[b];
  const uint8_t* Kb = (const uint8_t*)P.lv.ent_k + ((size_t)g * P.ent_head_stride + (size_t)row0 * kD) * 2;
  const uint8_t* Vb = (const uint8_t*)P.lv.ent_v + ((size_t)g * P.ent_head_stride + (size_t)row0 * kD) * 2;
  const uint32_t* mask = P.lv.zoom_mask + (size_t)bg * P.mask_words;
  const float scale2 = rsqrtf((float)kD) * kLog2e;

  uint32_t qf[4][4];
  load_q_frags(P.q + ((size_t)b * P.Hq + (size_t)g * G) * kD, G, gid, t4, qf);
  float m_run = -INFINITY, l_run = 0.f;
  // acc[s][w][2o + c] = O[head 2*t4 + c][dim 64s + 8gid + 2w + o]
  float acc[2][4][4];
#pragma unroll
  for (int s = 0; s < 2; ++s)
#pragma unroll
    for (int w = 0; w < 4; ++w) { acc[s][w][0] = 0.f; acc[s][w][1] = 0.f; acc[s][w][2] = 0.f; acc[s][w][3] = 0.f; }

  const int ntiles = (row_end - row_begin + 15) >> 4;
  uint4 kf[2][4], vf[4][2];
  auto load_k = [&](int t) {
    const int r0 = row_begin + t * 16;
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
      const int row = min(r0 + 8 * nt + gid, row_end - 1);
      const uint8_t* p = Kb + (size_t)row * (kD * 2) + t4 * 16;
#pragma unroll
      for (int j = 0; j < 4; ++j) kf[nt][j] = ldg16(p + j * 64);
    }
  };
  auto load_v = [&](int t) {
    const int r0 = row_begin + t * 16;
#pragma unroll
    for (int rr = 0; rr < 4; ++rr) {
      const int row = min(r0 + 2 * t4 + (rr & 1) + 8 * (rr >> 1), row_end - 1);
      const uint8_t* p = Vb + (size_t)row * (kD * 2) + gid * 16;
      vf[rr][0] = ldg16(p);
      vf[rr][1] = ldg16(p + 128);
    }
  };
  if (warp < ntiles) { load_k(warp); load_v(warp); }
  for (int t = warp; t < ntiles; t += kFW) {
    const int r0 = row_begin + t * 16;
    float sacc[2][4];
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
      sacc[nt][0] = sacc[nt][1] = sacc[nt][2] = sacc[nt][3] = 0.f;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        mma16816(sacc[nt], qf[j][0], qf[j][1], kf[nt][j].x, kf[nt][j].y);
        mma16816(sacc[nt], qf[j][2], qf[j][3], kf[nt][j].z, kf[nt][j].w);
      }
    }
    const bool more = (t + kFW) < ntiles;
    if (more) load_k(t + kFW);
    // logits in the base-2 domain with the entry bias (0 for pool tokens, ln|S| for coarse entries,
    // -inf for expanded spans and for rows past the item)
    float z[2][2];
    if (r0 + 16 <= min(A, row_end)) {     // warp-uniform fast path: all pool tokens
#pragma unroll
      for (int nt = 0; nt < 2; ++nt) { z[nt][0] = sacc[nt][0] * scale2; z[nt][1] = sacc[nt][1] * scale2; }
    } else {
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int row = r0 + 8 * nt + 2 * t4 + e;
          float bias = 0.f;
          if (row >= row_end) bias = -INFINITY;
          else if (row >= A) {
            const int s = row - A;
            bias = (__ldcg(mask + (s >> 5)) & (1u << (s & 31))) ? -INFINITY : P.cv.ln_len[span0 + s] * kLog2e;
          }
          z[nt][e] = fmaf(sacc[nt][e], scale2, bias);
        }
    }
    const float mx = quad_max(fmaxf(fmaxf(z[0][0], z[0][1]), fmaxf(z[1][0], z[1][1])));
    const float m_new = fmaxf(m_run, mx);
    const float m_safe = (m_new == -INFINITY) ? 0.f : m_new;
    if (__any_sync(0xffffffffu, m_new > m_run)) {
      const float corr = exp2f(m_run - m_safe);         // this lane's head is gid
      l_run *= corr;
      const float ca = __shfl_sync(0xffffffffu, corr, 8 * t4);       // head 2*t4
      const float cb = __shfl_sync(0xffffffffu, corr, 8 * t4 + 4);   // head 2*t4+1
#pragma unroll
      for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int w = 0; w < 4; ++w) { acc[s][w][0] *= ca; acc[s][w][1] *= cb; acc[s][w][2] *= ca; acc[s][w][3] *= cb; }
    }
    m_run = m_new;
    const float p00 = exp2f(z[0][0] - m_safe), p01 = exp2f(z[0][1] - m_safe);
    const float p10 = exp2f(z[1][0] - m_safe), p11 = exp2f(z[1][1] - m_safe);
    l_run += (p00 + p01) + (p10 + p11);
    uint32_t b0h, b0l, b1h, b1l;          // P^T fragments: n = head gid, k = tokens 2*t4+e (b0) and 8+2*t4+e (b1)
    split_bf16(p00, p01, b0h, b0l);
    split_bf16(p10, p11, b1h, b1l);
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      const uint32_t ra[4] = {vf[0][s].x, vf[0][s].y, vf[0][s].z, vf[0][s].w};
      const uint32_t rb[4] = {vf[1][s].x, vf[1][s].y, vf[1][s].z, vf[1][s].w};
      const uint32_t rc[4] = {vf[2][s].x, vf[2][s].y, vf[2][s].z, vf[2][s].w};
      const uint32_t rd[4] = {vf[3][s].x, vf[3][s].y, vf[3][s].z, vf[3][s].w};
#pragma unroll
      for (int w = 0; w < 4; ++w) {
        const uint32_t a0 = __byte_perm(ra[w], rb[w], 0x5410), a1 = __byte_perm(ra[w], rb[w], 0x7632);
        const uint32_t a2 = __byte_perm(rc[w], rd[w], 0x5410), a3 = __byte_perm(rc[w], rd[w], 0x7632);
        mma16816_full(acc[s][w], a0, a1, a2, a3, b0h, b1h);
        mma16816_full(acc[s][w], a0, a1, a2, a3, b0l, b1l);
      }
    }
    if (more) load_v(t + kFW);
  }
  l_run = quad_sum(l_run);
  if (gid < G && t4 == 0) { sm_ml[(warp * G + gid) * 2] = m_run; sm_ml[(warp * G + gid) * 2 + 1] = l_run; }
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    const int hh = 2 * t4 + c;
    if (hh < G) {
      float* o = sm_o + (warp * G + hh) * kD;
#pragma unroll
      for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int w = 0; w < 4; ++w) {
          o[64 * s + 8 * gid + 2 * w] = acc[s][w][c];
          o[64 * s + 8 * gid + 2 * w + 1] = acc[s][w][2 + c];
        }
    }
  }
  cta_merge_store<G>(sm_o, sm_ml, partial_out);
}

// ---------------------------------------------------------------------------------------------------
// a6: one expanded span, blob resident in shared memory; the CTA's warps split its 16-token chunks.
//   c = sigma_K o (Vt_K q) * log2e/sqrt(d)   (rows of Vt_K play the role of tokens in QK^T)
//   logits = U_K c  (= (U Sigma V^T q), Eq. 8 never materialised), p = 2^(z - m)
//   y = p^T U_V,   o += (sigma_V o y) V_V^T  accumulated into the warp's running (M, L, of)
// ---------------------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ void zoom_span_warp(const uint8_t* blob, const BlobDims& bd, int warp, int lane,
                                               const uint32_t (&qf)[4][4], float& M, float& L, float (&of)[16][4]) {
  const int gid = lane >> 2, t4 = lane & 3;
  const float* sK = (const float*)(blob + bd.off_sk);
  const float* sV = (const float*)(blob + bd.off_sv);
  const uint8_t* VtK = blob + bd.off_vtk;
  const uint8_t* VV = blob + bd.off_vv;
  const int nks = (bd.rkp + 15) >> 4, nvs = (bd.rvp + 15) >> 4;     // k-steps over the key / value rank
  const int ngrp = bd.lenp >> 4;
  if (warp >= ngrp) return;                                          // warp-uniform: nothing for this warp
  const float scale2 = rsqrtf((float)kD) * kLog2e;
  // 1. c
  uint32_t ckh[4][2], ckl[4][2];
#pragma unroll
  for (int ks = 0; ks < 4; ++ks) {
    ckh[ks][0] = ckh[ks][1] = ckl[ks][0] = ckl[ks][1] = 0u;
    if (ks < nks) {
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int nt = 2 * ks + u;
        float cf[4] = {0.f, 0.f, 0.f, 0.f};
        const int irow = pi_index(nt, gid);
        const bool have = irow < bd.rkp;     // rows past the padded rank do not exist: feed zeros
        const uint8_t* prow = VtK + (size_t)(have ? irow : 0) * (kD * 2) + t4 * 16;
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
          uint4 kv = make_uint4(0u, 0u, 0u, 0u);
          if (have) kv = *reinterpret_cast<const uint4*>(prow + jj * 64);
          mma16816(cf, qf[jj][0], qf[jj][1], kv.x, kv.y);
          mma16816(cf, qf[jj][2], qf[jj][3], kv.z, kv.w);
        }
        // columns 2*t4+e of n-tile nt are rank index pi(nt, 2*t4+e) = 16ks + 4*t4 + 2u + e
        const int i0 = 16 * ks + 4 * t4 + 2 * u;
        const float s0 = (i0 < bd.rkp) ? sK[i0] * scale2 : 0.f;
        const float s1 = (i0 + 1 < bd.rkp) ? sK[i0 + 1] * scale2 : 0.f;
        split_bf16(cf[0] * s0, cf[1] * s1, ckh[ks][u], ckl[ks][u]);
      }
    }
  }
  // 2. the warp's token chunks
  float m_s = -INFINITY, l_s = 0.f;
  float yf[8][4];
#pragma unroll
  for (int n = 0; n < 8; ++n) { yf[n][0] = yf[n][1] = yf[n][2] = yf[n][3] = 0.f; }
  for (int grp = warp; grp < ngrp; grp += kFW) {
    const uint8_t* UKc = blob + bd.off_chunks + (size_t)grp * bd.chunk_bytes;
    const uint8_t* UVtc = UKc + bd.uvt_in_chunk;
    float sacc[2][4];
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      sacc[u][0] = sacc[u][1] = sacc[u][2] = sacc[u][3] = 0.f;
      const uint8_t* prow = UKc + (size_t)pi_index(u, gid) * (bd.rkp * 2) + t4 * 8;
#pragma unroll
      for (int ks = 0; ks < 4; ++ks) {
        if (ks < nks) {
          uint2 bv = make_uint2(0u, 0u);
          if (16 * ks + 4 * t4 < bd.rkp) bv = *reinterpret_cast<const uint2*>(prow + ks * 32);
          mma16816(sacc[u], ckh[ks][0], ckh[ks][1], bv.x, bv.y);
          mma16816(sacc[u], ckl[ks][0], ckl[ks][1], bv.x, bv.y);
        }
      }
    }
    // this lane: head gid, tokens 16grp + 4*t4 + 2u + e
    float z[2][2];
#pragma unroll
    for (int u = 0; u < 2; ++u)
#pragma unroll
      for (int e = 0; e < 2; ++e) z[u][e] = (16 * grp + 4 * t4 + 2 * u + e < bd.len) ? sacc[u][e] : -INFINITY;
    const float mx = quad_max(fmaxf(fmaxf(z[0][0], z[0][1]), fmaxf(z[1][0], z[1][1])));
    const float m_new = fmaxf(m_s, mx);
    const float m_safe = (m_new == -INFINITY) ? 0.f : m_new;
    if (__any_sync(0xffffffffu, m_new > m_s)) {
      const float corr = exp2f(m_s - m_safe);
      l_s *= corr;
#pragma unroll
      for (int n = 0; n < 8; ++n) { yf[n][0] *= corr; yf[n][1] *= corr; }
    }
    m_s = m_new;
    const float p00 = exp2f(z[0][0] - m_safe), p01 = exp2f(z[0][1] - m_safe);
    const float p10 = exp2f(z[1][0] - m_safe), p11 = exp2f(z[1][1] - m_safe);
    l_s += (p00 + p01) + (p10 + p11);
    uint32_t a0h, a0l, a2h, a2l;
    split_bf16(p00, p01, a0h, a0l);     // tokens 4*t4 + {0,1}  <-> k = 2*t4 + e
    split_bf16(p10, p11, a2h, a2l);     // tokens 4*t4 + {2,3}  <-> k = 8 + 2*t4 + e
    // y += P U_V : B[k = token][n = i] read from the transposed factor UVt[i][token]
#pragma unroll
    for (int n = 0; n < 8; ++n) {
      if (n < 2 * nvs) {
        const int irow = pi_index(n, gid);
        uint2 bv = make_uint2(0u, 0u);
        if (irow < bd.rvp) bv = *reinterpret_cast<const uint2*>(UVtc + (size_t)irow * (kLenPad * 2) + t4 * 8);
        mma16816(yf[n], a0h, a2h, bv.x, bv.y);
        mma16816(yf[n], a0l, a2l, bv.x, bv.y);
      }
    }
  }
  // 3. fold the span into the warp's running state: of = of * 2^(M - M') + (sigma_V o y) V_V^T * 2^(m_s - M')
  const float M_new = fmaxf(M, m_s);
  const float M_safe = (M_new == -INFINITY) ? 0.f : M_new;
  const float c_old = exp2f(M - M_safe), c_new = exp2f(m_s - M_safe);
  L = fmaf(L, c_old, l_s * c_new);
  M = M_new;
#pragma unroll
  for (int nd = 0; nd < 16; ++nd) { of[nd][0] *= c_old; of[nd][1] *= c_old; }
  uint32_t yh[4][2], yl[4][2];          // yf[n][e] is head gid, rank index 16(n>>1) + 4*t4 + 2(n&1) + e
#pragma unroll
  for (int ks = 0; ks < 4; ++ks) {
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      yh[ks][u] = yl[ks][u] = 0u;
      if (ks < nvs) {
        const int i0 = 16 * ks + 4 * t4 + 2 * u;
        const float s0 = (i0 < bd.rvp) ? sV[i0] * c_new : 0.f;
        const float s1 = (i0 + 1 < bd.rvp) ? sV[i0 + 1] * c_new : 0.f;
        split_bf16(yf[2 * ks + u][0] * s0, yf[2 * ks + u][1] * s1, yh[ks][u], yl[ks][u]);
      }
    }
  }
#pragma unroll
  for (int nd = 0; nd < 16; ++nd) {
    const uint8_t* prow = VV + (size_t)(8 * nd + gid) * (bd.rvp * 2) + t4 * 8;
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      if (ks < nvs) {
        uint2 bv = make_uint2(0u, 0u);
        if (16 * ks + 4 * t4 < bd.rvp) bv = *reinterpret_cast<const uint2*>(prow + ks * 32);
        mma16816(of[nd], yh[ks][0], yh[ks][1], bv.x, bv.y);
        mma16816(of[nd], yl[ks][0], yl[ks][1], bv.x, bv.y);
      }
    }
  }
}

// wait until the plan of (b, g) has been published for this launch
__device__ __forceinline__ void wait_plan(const FusedParams& P, int bg, uint32_t epoch) {
  if (threadIdx.x == 0) {
    const uint32_t* f = (const uint32_t*)(P.ctrs + 2 + 3 * bg + 2);
    while (ld_acquire(f) != epoch) __nanosleep(64);
  }
  __syncthreads();
}

template <int G>
__device__ __forceinline__ void zoom_item(const FusedParams& P, const Item& I, uint8_t* dsm, Shared& S, float* sm_o,
                                          uint32_t (&phase)[2], float* __restrict__ partial_out) {
  const int bg = I.bg, b = bg / P.Hkv, g = bg % P.Hkv;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int gid = lane >> 2, t4 = lane & 3;
  const int n_zoom = __ldcg(P.plan_counts + 2 * bg);
  const int j0 = I.a, j1 = min(I.b, n_zoom);
  const int span0 = P.cv.seq_span_off[b];
  uint32_t qf[4][4];
  load_q_frags(P.q + ((size_t)b * P.Hq + (size_t)g * G) * kD, G, gid, t4, qf);
  float M = -INFINITY, L = 0.f;
  float of[16][4];
#pragma unroll
  for (int n = 0; n < 16; ++n) { of[n][0] = of[n][1] = of[n][2] = of[n][3] = 0.f; }

  auto issue = [&](int j) {            // thread 0 only
    const int buf = (j - j0) & 1;
    const int id = __ldcg(P.lv.item_span + (size_t)bg * P.kc + j);
    ZDesc d;
    d.valid = 0; d.miss = 0; d.len = 0; d.rr = 0; d.way = 0; d.bytes = 0;
    if (id >= 0) {
      const uint32_t it = __ldcg(P.lv.items + (size_t)bg * P.kc + j);
      const int gs = span0 + id;
      d.valid = 1;
      d.miss = (it >> 31) & 1;
      d.way = (int)(it & 0x7FFFFFFFu);
      d.rr = P.lv.dir_rank[(size_t)g * P.spans_cap + gs];
      d.len = P.cv.span_len[gs];
      const BlobDims bd = blob_dims(2, d.len, d.rr & 0xff, (d.rr >> 8) & 0xff);
      d.bytes = (uint32_t)bd.bytes;
      const uint8_t* src = d.miss ? P.host_arena + P.lv.dir_off[(size_t)g * P.spans_cap + gs]
                                  : P.lv.slots + ((size_t)bg * P.ways + d.way) * P.slot_bytes;
      fence_proxy_async();
      mbar_arrive_expect_tx(&S.bars[buf], d.bytes);
      bulk_g2s(dsm + (size_t)buf * P.smem_buf_stride, src, d.bytes, &S.bars[buf]);
    } else {
      mbar_arrive(&S.bars[buf]);
    }
    S.desc[buf] = d;
  };
  if (tid == 0) {
    if (j0 < j1) issue(j0);
    if (j0 + 1 < j1) issue(j0 + 1);
  }
  __syncthreads();                                 // descriptors visible
  for (int j = j0; j < j1; ++j) {
    const int buf = (j - j0) & 1;
    mbar_wait(&S.bars[buf], phase[buf]);
    phase[buf] ^= 1u;
    const ZDesc d = S.desc[buf];
    const uint8_t* blob = dsm + (size_t)buf * P.smem_buf_stride;
    if (d.valid) {
      const BlobDims bd = blob_dims(2, d.len, d.rr & 0xff, (d.rr >> 8) & 0xff);
      zoom_span_warp<G>(blob, bd, warp, lane, qf, M, L, of);
      if (d.miss) {                                // demand miss: the blob came over PCIe; keep it in its slot
        int4* dst = reinterpret_cast<int4*>(P.lv.slots + ((size_t)bg * P.ways + d.way) * P.slot_bytes);
        const int4* src = reinterpret_cast<const int4*>(blob);
        for (int i = tid; i < (int)(d.bytes >> 4); i += kFT) dst[i] = src[i];
      }
    }
    __syncthreads();                               // everyone is done with buf (and has read its descriptor)
    if (tid == 0 && j + 2 < j1) issue(j + 2);
    if (j + 2 < j1) __syncthreads();               // next descriptor visible (block-uniform condition)
  }
  // warp results -> shared memory -> one partial
  L = quad_sum(L);
  float* sm_ml = S.ml;
  if (gid < G) {
    if (t4 == 0) { sm_ml[(warp * G + gid) * 2] = M; sm_ml[(warp * G + gid) * 2 + 1] = L; }
    float* o = sm_o + (warp * G + gid) * kD;          // of[nd][c] is head gid, dimension 8*nd + 2*t4 + c
#pragma unroll
    for (int nd = 0; nd < 16; ++nd) { o[8 * nd + 2 * t4] = of[nd][0]; o[8 * nd + 2 * t4 + 1] = of[nd][1]; }
  }
  cta_merge_store<G>(sm_o, sm_ml, partial_out);
}

// ---------------------------------------------------------------------------------------------------
// a7: log-sum-exp merge of all partials of (b, g) -> out, lse.  Run by the last attention item of the
// group to finish.  Warp w takes partials p = w, w+4, ...; lane owns 4 output dimensions.
// ---------------------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ void combine_group(const FusedParams& P, int bg, uint8_t* dsm, float* sm_o) {
  const int b = bg / P.Hkv, g = bg % P.Hkv;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int p0 = P.bg_part_base[bg], n = P.bg_part_base[bg + 1] - p0;
  const float* parts = P.partials + (size_t)p0 * G * kPartStride;
  float* sh_w = reinterpret_cast<float*>(dsm);                 // [G][kCombineMaxParts] weights, then [G] L, [G] M
  float* sh_L = sh_w + G * kCombineMaxParts;
  float* sh_M = sh_L + SEKV_MAX_GROUP;
  __syncthreads();
  for (int hl = warp; hl < G; hl += kFW) {
    float mm = -INFINITY;
    for (int p = lane; p < n; p += 32) mm = fmaxf(mm, __ldcg(parts + ((size_t)p * G + hl) * kPartStride));
    mm = warp_max(mm);
    float ls = 0.f;
    for (int p = lane; p < n; p += 32) {
      const float* pp = parts + ((size_t)p * G + hl) * kPartStride;
      const float mp = __ldcg(pp);
      const float w = (mp == -INFINITY) ? 0.f : exp2f(mp - mm);
      sh_w[hl * kCombineMaxParts + p] = w;
      ls = fmaf(__ldcg(pp + 1), w, ls);
    }
    ls = warp_sum(ls);
    if (lane == 0) { sh_L[hl] = ls; sh_M[hl] = mm; }
  }
  __syncthreads();
  float4 acc[G];
#pragma unroll
  for (int hl = 0; hl < G; ++hl) acc[hl] = make_float4(0.f, 0.f, 0.f, 0.f);
  for (int p = warp; p < n; p += kFW) {
#pragma unroll
    for (int hl = 0; hl < G; ++hl) {
      const float w = sh_w[hl * kCombineMaxParts + p];
      const float4 v = __ldcg(reinterpret_cast<const float4*>(parts + ((size_t)p * G + hl) * kPartStride + 4) + lane);
      acc[hl].x = fmaf(v.x, w, acc[hl].x); acc[hl].y = fmaf(v.y, w, acc[hl].y);
      acc[hl].z = fmaf(v.z, w, acc[hl].z); acc[hl].w = fmaf(v.w, w, acc[hl].w);
    }
  }
#pragma unroll
  for (int hl = 0; hl < G; ++hl) reinterpret_cast<float4*>(sm_o + (warp * G + hl) * kD)[lane] = acc[hl];
  __syncthreads();
  for (int o = tid; o < G * kD; o += kFT) {
    const int hl = o / kD, d = o % kD;
    float v = 0.f;
#pragma unroll
    for (int w = 0; w < kFW; ++w) v += sm_o[(w * G + hl) * kD + d];
    const float Ls = sh_L[hl];
    const float res = Ls > 0.f ? v / Ls : 0.f;
    const size_t oi = ((size_t)b * P.Hq + (size_t)g * G + hl) * kD + d;
    if (P.out_bf16) reinterpret_cast<__nv_bfloat16*>(P.out)[oi] = __float2bfloat16_rn(res);
    else reinterpret_cast<float*>(P.out)[oi] = res;
    if (P.lse && d == 0) P.lse[b * P.Hq + g * G + hl] = Ls > 0.f ? (sh_M[hl] + log2f(Ls)) * kLn2 : -INFINITY;
  }
  __syncthreads();
}

// the partial of an attention item is written; the last item of the group combines
template <int G>
__device__ __forceinline__ void attn_item_done(const FusedParams& P, int bg, uint8_t* dsm, Shared& S, float* sm_o) {
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    const int expected = P.bg_part_base[bg + 1] - P.bg_part_base[bg];
    int* ctr = P.ctrs + 2 + 3 * bg + 1;
    const int old = atomicAdd(ctr, 1);
    S.flag = (old == expected - 1);
    if (S.flag) *ctr = 0;
  }
  __syncthreads();
  if (S.flag) {
    __threadfence();
    combine_group<G>(P, bg, dsm, sm_o);
  }
}

// ---------------------------------------------------------------------------------------------------
// a3: bitonic sort (descending) of n 64-bit keys in shared memory
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void bitonic_sort_desc(unsigned long long* keys, int n) {
  for (int size = 2; size <= n; size <<= 1) {
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int i = threadIdx.x; i < (n >> 1); i += kFT) {
        const int lo = ((i & ~(stride - 1)) << 1) | (i & (stride - 1));
        const int hi = lo | stride;
        const bool desc = ((lo & size) == 0);
        const unsigned long long a = keys[lo], c = keys[hi];
        if ((a < c) == desc) { keys[lo] = c; keys[hi] = a; }
      }
      __syncthreads();
    }
  }
}

// block-wide exclusive scan of one flag per thread; returns this thread's offset, total in *total
__device__ __forceinline__ int block_scan_flag(bool f, Shared& S, int* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned bal = __ballot_sync(0xffffffffu, f);
  __syncthreads();
  if (lane == 0) S.scan[warp] = __popc(bal);
  __syncthreads();
  int base = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < kFW; ++w) { const int c = S.scan[w]; if (w < warp) base += c; tot += c; }
  *total = tot;
  return base + __popc(bal & ((1u << lane) - 1u));
}

// ---------------------------------------------------------------------------------------------------
// a4: residency plan of (b, g) (one CTA).  The device factor cache of a (layer, sequence, kv head) is
// `ways` slots with a tag (span id) and a stamp (step of last use).  The first n_zoom entries of
// sh_ids are this step's zoom set: resident ones are hits, the others are demand misses and take the
// least-recently-used slots not needed by this step.  Entries n_zoom .. n_cand-1 are prefetch
// candidates (the next-best spans by routing score): the non-resident ones get a slot too and are
// copied by the side-stream prefetch kernel after this layer's kernel.  Also: zoom bit-mask for the
// coarse items (an expanded span's coarse entry is replaced by its tokens),
// de-duplication of caller-supplied ids, statistics.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void plan_block(const FusedParams& P, int bg, uint8_t* dsm, Shared& S, int n_zoom, int n_cand,
                                           bool dedupe, uint32_t epoch) {
  const int b = bg / P.Hkv, g = bg % P.Hkv, tid = threadIdx.x;
  const int span0 = P.cv.seq_span_off[b];
  const int m = P.cv.seq_span_off[b + 1] - span0;
  const int ways = P.ways;
  int32_t* sh_ids = reinterpret_cast<int32_t*>(dsm + P.sm_ids);
  int16_t* way_of = reinterpret_cast<int16_t*>(dsm + P.sm_wayof);
  int32_t* sh_tag = reinterpret_cast<int32_t*>(dsm + P.sm_tags);
  uint32_t* sh_stamp = reinterpret_cast<uint32_t*>(sh_tag + ways);
  int32_t* sh_victim = reinterpret_cast<int32_t*>(sh_stamp + ways);
  uint32_t* sh_mask = reinterpret_cast<uint32_t*>(dsm + P.sm_mask);
  int32_t* tags = P.lv.tags + (size_t)bg * ways;
  uint32_t* stamps = P.lv.stamps + (size_t)bg * ways;
  uint32_t* items = P.lv.items + (size_t)bg * P.kc;
  int32_t* item_span = P.lv.item_span + (size_t)bg * P.kc;
  const uint32_t cur = epoch;
  for (int w = tid; w < P.mask_words; w += kFT) sh_mask[w] = 0u;
  for (int s = tid; s < m; s += kFT) way_of[s] = (int16_t)-1;
  for (int w = tid; w < ways; w += kFT) { sh_tag[w] = tags[w]; sh_stamp[w] = stamps[w]; }
  __syncthreads();
  for (int w = tid; w < ways; w += kFT) { const int t = sh_tag[w]; if (t >= 0 && t < m) way_of[t] = (int16_t)w; }
  __syncthreads();
  unsigned long long n_hit = 0, n_miss = 0, bytes_algo = 0, bytes_h2d = 0, n_pf = 0, bytes_pf = 0;
  // pass 1: validate / de-duplicate, zoom mask, residency lookup
  for (int j = tid; j < n_cand; j += kFT) {
    int id = sh_ids[j];
    if (id < 0 || id >= m) id = -1;
    const bool zoom = j < n_zoom;
    if (id >= 0 && zoom) {
      const uint32_t bit = 1u << (id & 31);
      const uint32_t old = atomicOr(&sh_mask[id >> 5], bit);
      if (dedupe && (old & bit)) id = -1;                      // duplicate of an id seen before: dropped
    }
    int way = -1;
    if (id >= 0) {
      way = way_of[id];
      if (way >= 0) sh_stamp[way] = cur;
      const int rr = P.lv.dir_rank[(size_t)g * P.spans_cap + span0 + id];
      const int rk = rr & 0xff, rv = (rr >> 8) & 0xff;
      const int len = P.cv.span_len[span0 + id];
      const unsigned long long bb = blob_dims(2, len, rk, rv).bytes;
      if (zoom) {
        bytes_algo += (unsigned long long)(rk + rv) * (len + kD) * 2 + 4ull * (rk + rv);
        if (way >= 0) ++n_hit; else { ++n_miss; bytes_h2d += bb; }
      } else if (way < 0) { ++n_pf; bytes_pf += bb; }
    }
    sh_ids[j] = id;
    item_span[j] = id;
    items[j] = (way >= 0) ? (uint32_t)way : 0xFFFFFFFFu;
  }
  __syncthreads();
  // victims: ways not used by this step, oldest stamp first (ties to the lower way)
  for (int w = tid; w < ways; w += kFT) {
    if (sh_stamp[w] != cur) {
      int rank = 0;
      const uint32_t mine = sh_stamp[w];
      for (int v = 0; v < ways; ++v) {
        const uint32_t o = sh_stamp[v];
        rank += (o != cur) && (o < mine || (o == mine && v < w));
      }
      sh_victim[rank] = w;
    }
  }
  __syncthreads();
  // pass 2: misses take victims in item order
  int miss_base = 0;
  for (int j0 = 0; j0 < n_cand; j0 += kFT) {
    const int j = j0 + tid;
    const bool miss = (j < n_cand) && sh_ids[j] >= 0 && items[j] == 0xFFFFFFFFu;
    int tot;
    const int off = block_scan_flag(miss, S, &tot);
    if (miss) {
      const int way = sh_victim[miss_base + off];
      sh_tag[way] = sh_ids[j];
      sh_stamp[way] = cur;
      items[j] = (uint32_t)way | 0x80000000u;
    }
    miss_base += tot;
  }
  __syncthreads();
  for (int w = tid; w < ways; w += kFT) { tags[w] = sh_tag[w]; stamps[w] = sh_stamp[w]; }
  uint32_t* gmask = P.lv.zoom_mask + (size_t)bg * P.mask_words;
  for (int w = tid; w < P.mask_words; w += kFT) gmask[w] = sh_mask[w];
  if (tid == 0) { P.plan_counts[2 * bg] = n_zoom; P.plan_counts[2 * bg + 1] = n_cand; }
  // statistics
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    n_hit += __shfl_xor_sync(0xffffffffu, n_hit, o);
    n_miss += __shfl_xor_sync(0xffffffffu, n_miss, o);
    bytes_algo += __shfl_xor_sync(0xffffffffu, bytes_algo, o);
    bytes_h2d += __shfl_xor_sync(0xffffffffu, bytes_h2d, o);
    n_pf += __shfl_xor_sync(0xffffffffu, n_pf, o);
    bytes_pf += __shfl_xor_sync(0xffffffffu, bytes_pf, o);
  }
  if ((tid & 31) == 0) {
    if (n_hit) atomicAdd(&P.stats[ST_HITS], n_hit);
    if (n_miss) atomicAdd(&P.stats[ST_MISSES], n_miss);
    if (n_hit + n_miss) { atomicAdd(&P.stats[ST_ZOOMED], n_hit + n_miss); atomicAdd(&P.stats[ST_SKIPPED], n_hit + n_miss); }
    if (bytes_algo) atomicAdd(&P.stats[ST_FACTOR_ALGO], bytes_algo);
    if (bytes_h2d + bytes_pf) atomicAdd(&P.stats[ST_H2D], bytes_h2d + bytes_pf);
    if (n_pf) atomicAdd(&P.stats[ST_PREFETCHED], n_pf);
  }
  __threadfence();
  __syncthreads();
  if (tid == 0) st_release((uint32_t*)(P.ctrs + 2 + 3 * bg + 2), epoch);
}

// ---------------------------------------------------------------------------------------------------
// a1-a3: one chunk of spans of (b, g)
// ---------------------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ void route_item(const FusedParams& P, const Item& I, uint8_t* dsm, Shared& S, uint32_t epoch) {
  const int bg = I.bg, b = bg / P.Hkv, g = bg % P.Hkv, tid = threadIdx.x;
  const int span0 = P.cv.seq_span_off[b];
  const int m = P.cv.seq_span_off[b + 1] - span0;
  const int dp = P.dp;
  unsigned long long* gkeys = P.keys + (size_t)bg * P.sort_n;
  if (P.mode & FM_ROUTE) {
    float* sh_q = reinterpret_cast<float*>(dsm);               // [G][128]
    float* sh_qp = sh_q + G * kD;                              // [G][dp]
    const __nv_bfloat16* q = P.q + ((size_t)b * P.Hq + (size_t)g * G) * kD;
    for (int o = tid; o < G * kD; o += kFT) sh_q[o] = __bfloat162float(q[o]);
    __syncthreads();
    const __nv_bfloat16* W = (const __nv_bfloat16*)P.lv.W;
    for (int o = tid; o < G * dp; o += kFT) {                  // Eq. 4: one thread per (head, j)
      const int hl = o / dp, j = o % dp;
      const __nv_bfloat16* wr = W + ((size_t)(g * G + hl) * dp + j) * kD;
      float acc = 0.f;
#pragma unroll 4
      for (int d = 0; d < kD; d += 8) {
        const uint4 v = *reinterpret_cast<const uint4*>(wr + d);
        const uint32_t ww[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          acc = fmaf(__uint_as_float(ww[e] << 16), sh_q[hl * kD + d + 2 * e], acc);
          acc = fmaf(__uint_as_float(ww[e] & 0xffff0000u), sh_q[hl * kD + d + 2 * e + 1], acc);
        }
      }
      sh_qp[o] = acc;
    }
    __syncthreads();
    const float inv_sqrt_dp = rsqrtf((float)dp);
    const __nv_bfloat16* route = (const __nv_bfloat16*)P.lv.route;
    for (int s = I.a + tid; s < I.b; s += kFT) {
      const float lnl = P.cv.ln_len[span0 + s];
      float X = -INFINITY;
      bool elig = (P.tau == nullptr);
#pragma unroll
      for (int hl = 0; hl < G; ++hl) {
        const int h = g * G + hl;
        const __nv_bfloat16* kr = route + (size_t)h * P.route_head_stride + (size_t)(span0 + s) * dp;
        float acc = 0.f;
        for (int j = 0; j < dp; j += 8) {
          const uint4 v = ldg16(kr + j);
          const uint32_t ww[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            acc = fmaf(__uint_as_float(ww[e] << 16), sh_qp[hl * dp + j + 2 * e], acc);
            acc = fmaf(__uint_as_float(ww[e] & 0xffff0000u), sh_qp[hl * dp + j + 2 * e + 1], acc);
          }
        }
        const float x = fmaf(acc, inv_sqrt_dp, lnl);           // Eq. 5, pre-sigmoid logit
        const float a = 1.f / (1.f + __expf(-x));
        if (P.logits_out) P.logits_out[(size_t)h * P.m_tot + span0 + s] = x;
        if (P.alpha_out) P.alpha_out[(size_t)h * P.m_tot + span0 + s] = a;
        if (P.tau != nullptr && a > P.tau[h]) elig = true;     // Eq. 9
        X = fmaxf(X, x);
      }
      gkeys[s] = elig ? (((unsigned long long)order_key(X) << 32) | (unsigned long long)(0xFFFFFFFFu - (uint32_t)s)) : 0ull;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) {
      int* ctr = P.ctrs + 2 + 3 * bg;
      const int old = atomicAdd(ctr, 1);
      S.flag = (old == P.bg_route_items[bg] - 1);
      if (S.flag) *ctr = 0;
    }
    __syncthreads();
    if (!S.flag) return;
    __threadfence();
    // last chunk of the group: top-k
    unsigned long long* keys = reinterpret_cast<unsigned long long*>(dsm);
    int my = 0;
    for (int s = tid; s < P.sort_n; s += kFT) {
      const unsigned long long k = (s < m) ? __ldcg(gkeys + s) : 0ull;
      keys[s] = k;
      my += (k != 0ull);
    }
    my = (int)warp_sum((float)my);                 // exact for counts < 2^24
    __syncthreads();
    if ((tid & 31) == 0) S.scan[tid >> 5] = my;
    __syncthreads();
    int n_elig = 0;
#pragma unroll
    for (int w = 0; w < kFW; ++w) n_elig += S.scan[w];
    bitonic_sort_desc(keys, P.sort_n);
    int cnt = P.k < 0 ? n_elig : min(P.k, n_elig);
    cnt = min(cnt, P.k_cap);
    int n_cand = cnt;
    if (P.k >= 0 && (P.mode & FM_ATTN)) n_cand = min(min(cnt + P.prefetch, n_elig), P.kc);
    int32_t* sh_ids = reinterpret_cast<int32_t*>(dsm + P.sm_ids);
    int32_t* my_ids = P.ids + (size_t)bg * max(P.k_cap, 1);
    for (int j = tid; j < max(P.k_cap, n_cand); j += kFT) {
      const int id = j < n_cand ? (int32_t)(0xFFFFFFFFu - (uint32_t)(keys[j] & 0xFFFFFFFFull)) : -1;
      if (j < n_cand) sh_ids[j] = id;
      if (j < P.k_cap) my_ids[j] = j < cnt ? id : -1;
    }
    if (tid == 0) P.count[bg] = cnt;
    __syncthreads();
    if (P.mode & FM_ATTN) plan_block(P, bg, dsm, S, cnt, n_cand, false, epoch);
  } else {
    // caller-supplied zoom set (sekv_decode_attn): the group's first chunk item runs the plan
    if (I.a != 0) return;
    int cnt = 0;
    if (P.ids != nullptr && P.count != nullptr) cnt = max(0, min(P.count[bg], P.k_cap));
    int32_t* sh_ids = reinterpret_cast<int32_t*>(dsm + P.sm_ids);
    const int32_t* src = P.ids + (size_t)bg * max(P.k_cap, 1);
    for (int j = tid; j < cnt; j += kFT) sh_ids[j] = src[j];
    __syncthreads();
    plan_block(P, bg, dsm, S, cnt, cnt, true, epoch);
  }
}

template <int G>
__global__ void __launch_bounds__(kFT, 3) fused_layer_kernel(const __grid_constant__ FusedParams P) {
  extern __shared__ __align__(128) uint8_t dsm[];
  __shared__ Shared S;
  __shared__ __align__(16) float sm_o[kFW * G * kD];
  const int tid = threadIdx.x;
  const uint32_t epoch = *reinterpret_cast<volatile const uint32_t*>(P.lv.layer_step) + 1u;
  if (tid == 0) {
    mbar_init(&S.bars[0], 1);
    mbar_init(&S.bars[1], 1);
    mbar_fence_init();
  }
  __syncthreads();
  uint32_t phase[2] = {0u, 0u};
  for (;;) {
    if (tid == 0) S.item = atomicAdd(P.ctrs, 1);
    __syncthreads();
    const int it = S.item;
    __syncthreads();
    if (it >= P.n_items) break;
    const Item I = P.items[it];
    if (I.kind == IT_ROUTE) {
      route_item<G>(P, I, dsm, S, epoch);
      __syncthreads();
      continue;
    }
    float* part = P.partials + ((size_t)P.bg_part_base[I.bg] + I.part) * G * kPartStride;
    if (I.kind == IT_POOL) {
      rows_item<G>(P, I.bg, I.a, I.b, sm_o, S.ml, part);
    } else if (I.kind == IT_COARSE) {
      wait_plan(P, I.bg, epoch);
      rows_item<G>(P, I.bg, I.a, I.b, sm_o, S.ml, part);
    } else {
      wait_plan(P, I.bg, epoch);
      zoom_item<G>(P, I, dsm, S, sm_o, phase, part);
    }
    attn_item_done<G>(P, I.bg, dsm, S, sm_o);
  }
  // last CTA out re-arms the queue and advances the layer's step stamp
  if (tid == 0) {
    __threadfence();
    const int old = atomicAdd(P.ctrs + 1, 1);
    if (old == (int)gridDim.x - 1) {
      P.ctrs[0] = 0;
      P.ctrs[1] = 0;
      if (P.mode & FM_ATTN) {
        *P.lv.layer_step = epoch;
        atomicAdd(&P.stats[ST_LAYER_STEPS], 1ull);
      }
      __threadfence();
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// a4, side stream: copy the prefetch candidates that the plan gave a slot (items n_zoom .. n_cand-1 with
// the miss bit) from the pinned-host store into the device factor cache.  One warp per candidate; lane 0
// drives two bulk copies through a shared-memory bounce buffer (host -> smem over PCIe, smem -> slot).
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32) prefetch_kernel(CsrView cv, LayerView lv, const int32_t* __restrict__ plan_counts,
                                                      int kc, int Hkv, int ways, int spans_cap, int64_t slot_bytes,
                                                      const uint8_t* __restrict__ host_arena) {
  extern __shared__ __align__(128) uint8_t buf[];
  __shared__ uint64_t bar;
  const int bg = blockIdx.y, b = bg / Hkv, g = bg % Hkv;
  const int j = plan_counts[2 * bg] + blockIdx.x;
  if (j >= plan_counts[2 * bg + 1]) return;
  const int id = lv.item_span[(size_t)bg * kc + j];
  const uint32_t it = lv.items[(size_t)bg * kc + j];
  if (id < 0 || !(it & 0x80000000u)) return;
  if (threadIdx.x == 0) {
    const int way = (int)(it & 0x7FFFFFFFu);
    const int gs = cv.seq_span_off[b] + id;
    const int rr = lv.dir_rank[(size_t)g * spans_cap + gs];
    const uint32_t bytes = (uint32_t)blob_dims(2, cv.span_len[gs], rr & 0xff, (rr >> 8) & 0xff).bytes;
    mbar_init(&bar, 1);
    mbar_fence_init();
    mbar_arrive_expect_tx(&bar, bytes);
    bulk_g2s(buf, host_arena + lv.dir_off[(size_t)g * spans_cap + gs], bytes, &bar);
    mbar_wait(&bar, 0u);
    fence_proxy_async();
    bulk_s2g(lv.slots + ((size_t)bg * ways + way) * slot_bytes, buf, bytes);
    bulk_commit();
    bulk_wait_all();
  }
}

}  // namespace

// ---------------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------------
size_t fused_plan_smem(const sekv_handle* h, FusedParams* P) {
  const sekv_config& c = h->cfg;
  const int kc = std::max(c.k_cap, 1) + std::max(c.prefetch, 0);
  size_t o = (size_t)h->sort_n * 8;
  o = round_up_sz(o, 16); P->sm_ids = (int)o; o += (size_t)kc * 4;
  o = round_up_sz(o, 16); P->sm_wayof = (int)o; o += (size_t)round_up(std::max(h->max_m, 1), 8) * 2;
  o = round_up_sz(o, 16); P->sm_tags = (int)o; o += (size_t)c.cache_ways * 12;
  o = round_up_sz(o, 16); P->sm_mask = (int)o; o += (size_t)h->mask_words * 4;
  return o;
}

template <int G>
static cudaError_t launch_fused_g(sekv_handle* h, const FusedParams& P, size_t smem, int grid, cudaStream_t s) {
  static size_t configured = 0;
  if (smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(fused_layer_kernel<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  fused_layer_kernel<G><<<grid, kFT, smem, s>>>(P);
  return cudaGetLastError();
}

template <int G>
static int fused_occupancy_g(size_t smem) {
  int n = 0;
  cudaFuncSetAttribute(fused_layer_kernel<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, fused_layer_kernel<G>, kFT, smem);
  return n;
}

size_t fused_smem_bytes(const sekv_handle* h, FusedParams* P) {
  const sekv_config& c = h->cfg;
  FusedParams tmp;
  if (!P) P = &tmp;
  size_t need = fused_plan_smem(h, P);
  const size_t slotp = round_up_sz((size_t)h->lay.slot_bytes, 128);
  P->smem_buf_stride = (int64_t)slotp;
  if (c.k_cap > 0) need = std::max(need, 2 * slotp);
  need = std::max(need, (size_t)(h->G * kCombineMaxParts + 2 * SEKV_MAX_GROUP) * 4);
  need = std::max(need, (size_t)h->G * (kD + c.route_dim) * 4);
  return round_up_sz(need, 128);
}

int fused_occupancy(const sekv_handle* h) {
  const size_t smem = fused_smem_bytes(h, nullptr);
  switch (h->G) {
    case 1: return fused_occupancy_g<1>(smem); case 2: return fused_occupancy_g<2>(smem);
    case 3: return fused_occupancy_g<3>(smem); case 4: return fused_occupancy_g<4>(smem);
    case 5: return fused_occupancy_g<5>(smem); case 6: return fused_occupancy_g<6>(smem);
    case 7: return fused_occupancy_g<7>(smem); case 8: return fused_occupancy_g<8>(smem);
  }
  return 0;
}

cudaError_t launch_fused(sekv_handle* h, int layer, int mode, const void* q, const float* tau, int k, float* logits,
                         float* alpha, int32_t* ids, int32_t* count, void* out, float* lse, cudaStream_t s) {
  const sekv_config& c = h->cfg;
  FusedParams P;
  memset(&P, 0, sizeof(P));
  P.cv = csr_view(h);
  P.lv = layer_view(h, layer);
  P.q = (const __nv_bfloat16*)q; P.tau = tau; P.logits_out = logits; P.alpha_out = alpha;
  P.ids = ids; P.count = count; P.out = out; P.lse = lse;
  P.items = (const Item*)ws(h, h->F.off_items_sched);
  P.n_items = (mode & FM_ATTN) ? h->n_items : h->n_route_items;
  P.bg_part_base = (const int32_t*)ws(h, h->F.off_bg_part);
  P.bg_route_items = (const int32_t*)ws(h, h->F.off_bg_route);
  P.partials = (float*)ws(h, h->F.off_partials1);
  P.keys = (unsigned long long*)ws(h, h->F.off_keys);
  P.ctrs = (int32_t*)ws(h, h->F.off_ctrs) + (size_t)layer * h->F.ctrs_per_layer;
  P.plan_counts = (int32_t*)ws(h, h->F.off_plan_counts) + (size_t)layer * c.max_seqs * c.n_kv_heads * 2;
  P.stats = (unsigned long long*)ws(h, h->F.off_stats);
  P.host_arena = h->host_dev;
  P.mode = mode; P.k = k; P.k_cap = c.k_cap; P.prefetch = std::max(c.prefetch, 0);
  P.kc = std::max(c.k_cap, 1) + std::max(c.prefetch, 0);
  P.Hq = c.n_q_heads; P.Hkv = c.n_kv_heads; P.dp = c.route_dim; P.ways = c.cache_ways;
  P.mask_words = h->mask_words; P.spans_cap = (int)h->lay.spans_cap; P.m_tot = h->m_tot; P.sort_n = h->sort_n;
  P.out_bf16 = c.out_dtype == SEKV_BF16;
  P.slot_bytes = h->lay.slot_bytes;
  P.ent_head_stride = (size_t)h->lay.rows_cap * kD;
  P.route_head_stride = (size_t)h->lay.spans_cap * c.route_dim;
  const size_t smem = fused_smem_bytes(h, &P);
  const int grid = std::max(1, std::min(P.n_items, h->fused_grid));
  cudaError_t e;
  switch (h->G) {
    case 1: e = launch_fused_g<1>(h, P, smem, grid, s); break;
    case 2: e = launch_fused_g<2>(h, P, smem, grid, s); break;
    case 3: e = launch_fused_g<3>(h, P, smem, grid, s); break;
    case 4: e = launch_fused_g<4>(h, P, smem, grid, s); break;
    case 5: e = launch_fused_g<5>(h, P, smem, grid, s); break;
    case 6: e = launch_fused_g<6>(h, P, smem, grid, s); break;
    case 7: e = launch_fused_g<7>(h, P, smem, grid, s); break;
    case 8: e = launch_fused_g<8>(h, P, smem, grid, s); break;
    default: return cudaErrorInvalidValue;
  }
  h->launches += 1;
  return e;
}

cudaError_t launch_prefetch(sekv_handle* h, int layer, cudaStream_t s) {
  const sekv_config& c = h->cfg;
  if (c.prefetch <= 0 || c.k_cap <= 0) return cudaSuccess;
  static size_t configured = 0;
  const size_t smem = round_up_sz((size_t)h->lay.slot_bytes, 128);
  if (smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(prefetch_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  dim3 grid(c.prefetch, h->n_seqs * c.n_kv_heads);
  const int32_t* pc = (const int32_t*)ws(h, h->F.off_plan_counts) + (size_t)layer * c.max_seqs * c.n_kv_heads * 2;
  prefetch_kernel<<<grid, 32, smem, s>>>(csr_view(h), layer_view(h, layer), pc, std::max(c.k_cap, 1) + c.prefetch,
                                         c.n_kv_heads, c.cache_ways, (int)h->lay.spans_cap, h->lay.slot_bytes, h->host_dev);
  h->launches += 1;
  return cudaGetLastError();
}

}  // namespace sekv
