// a5 / a6 for bf16 storage: split-K flash-decode on the warp-level tensor-core path.
//
// The work is HBM-bound streaming with G <= 8 query heads per kv head, so there is no M >= 64 tile for
// tcgen05; what matters is that every stored byte is read once, fully coalesced, with as few issue
// slots per byte as possible.  The G heads of a group are the (padded) 16 rows of an
// mma.sync.m16n8k16 A operand; K rows, V rows and factor rows go from global memory straight into B
// fragments (no shared-memory staging, no bank conflicts), using the freedom to permute the
// contraction index consistently on both operands:
//
//   QK^T : lane (gid = lane/4, t4 = lane%4) loads 16-byte chunk (t4 + 4j) of the K row of token gid;
//          its four 32-bit words are the (b0,b1) pairs of two k-steps; Q is loaded the same way.
//   P V  : computed transposed, O^T = V^T P^T (M = 16 dims, N = 8 heads, K = 16 tokens): the C fragment
//          of S (row = head gid, cols = tokens 2*t4, 2*t4+1) IS the B fragment of P^T (n = gid,
//          k = 2*t4, 2*t4+1), so no data movement is needed between the two products.  Lane loads
//          chunk (gid + 8s) of rows 2*t4, 2*t4+1, 2*t4+8, 2*t4+9 of V and builds the token-pair A
//          fragments with one PRMT per word; rows gid / gid+8 of m-tile (s,w) are dimensions
//          64s + 8gid + 2w and + 1.
//   P (fp32) is split into bf16 hi + lo parts and multiplied twice, so probabilities carry ~16 bits.
//
// Stage 2 applies the query through the factored form with the same machinery:
//   c = Q Vt_K^T (like QK^T with the r rows of Vt_K as "tokens"), logits = (sigma_K o c) U_K^T,
//   y = P U_V, o = (sigma_V o y) V_V^T; each factor is stored with its contraction index contiguous
//   (blob layout, sekv_internal.cuh).
#include "sekv_internal.cuh"

namespace sekv {

namespace {

__device__ __forceinline__ void mma16816(float (&c)[4], uint32_t a0, uint32_t a2, uint32_t b0, uint32_t b1) {
  // rows 8..15 of A (a1, a3) are always zero: the group's heads occupy rows 0..G-1
  const uint32_t z = 0u;
  asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a0), "r"(z), "r"(a2), "r"(z), "r"(b0), "r"(b1));
}

// general form (all four A registers): used for O^T = V^T P^T where the 16 rows are dimensions
__device__ __forceinline__ void mma16816_full(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                              uint32_t b0, uint32_t b1) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

__device__ __forceinline__ uint4 ldg16(const void* p) {
  uint4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ uint2 ldg8(const void* p) {
  uint2 v;
  asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
  return v;
}

// bf16x2 with `lo` in the low half (lower k index) and `hi` in the high half
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t d;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
  return d;
}
// x = hi + lo with both parts bf16: ~16 significant bits survive the tensor-core multiply
__device__ __forceinline__ void split_bf16(float x0, float x1, uint32_t& hi, uint32_t& lo) {
  hi = pack_bf16(x0, x1);
  const float h0 = __uint_as_float(hi << 16), h1 = __uint_as_float(hi & 0xffff0000u);
  lo = pack_bf16(x0 - h0, x1 - h1);
}

__device__ __forceinline__ float quad_max(float v) {
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 1));
  return fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 2));
}
__device__ __forceinline__ float quad_sum(float v) {
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  return v + __shfl_xor_sync(0xffffffffu, v, 2);
}

// row permutation that makes a C fragment's columns line up with the next A fragment's k indices
// when the consumer loads 8 contiguous bytes (4 bf16) per lane: n-tile nt, column n -> index
__device__ __forceinline__ int pi_index(int nt, int n) { return 16 * (nt >> 1) + 4 * (n >> 1) + 2 * (nt & 1) + (n & 1); }

// Merge the warps' partials of one CTA in shared memory and write one partial per head.
// sm_o: [NW][G][128], sm_ml: [NW][G][2]
template <int G, int NW>
__device__ __forceinline__ void cta_merge_store(float* sm_o, float* sm_ml, float* __restrict__ out) {
  __syncthreads();
  for (int o = threadIdx.x; o < G * kD; o += NW * 32) {
    const int h = o / kD, d = o % kD;
    float mm = -INFINITY;
#pragma unroll
    for (int w = 0; w < NW; ++w) mm = fmaxf(mm, sm_ml[(w * G + h) * 2]);
    float ls = 0.f, os = 0.f;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      const float mw = sm_ml[(w * G + h) * 2];
      const float c = (mw == -INFINITY) ? 0.f : exp2f(mw - mm);
      ls = fmaf(sm_ml[(w * G + h) * 2 + 1], c, ls);
      os = fmaf(sm_o[(w * G + h) * kD + d], c, os);
    }
    if (d == 0) { out[h * kPartStride] = mm; out[h * kPartStride + 1] = ls; }
    out[h * kPartStride + 4 + d] = os;
  }
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// Stage 1
// ---------------------------------------------------------------------------------------------
template <int G, int NW>
__global__ void __launch_bounds__(NW * 32, (NW == 4) ? 3 : 1)
stage1_mma_kernel(CsrView cv, LayerView lv, const Chunk* __restrict__ chunks, const __nv_bfloat16* __restrict__ q,
                  int Hq, int Hkv, size_t ent_head_stride, int mask_words, float* __restrict__ partials) {
  __shared__ float sm_o[NW * G * kD];
  __shared__ float sm_ml[NW * G * 2];
  const Chunk ck = chunks[blockIdx.x];
  const int b = ck.bg / Hkv, g = ck.bg % Hkv;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int gid = lane >> 2, t4 = lane & 3;
  const int A = cv.seq_pool_cnt[b];
  const int row0 = cv.seq_row_off[b];
  const int span0 = cv.seq_span_off[b];
  const uint8_t* Kb = (const uint8_t*)lv.ent_k + ((size_t)g * ent_head_stride + (size_t)row0 * kD) * 2;
  const uint8_t* Vb = (const uint8_t*)lv.ent_v + ((size_t)g * ent_head_stride + (size_t)row0 * kD) * 2;
  const uint32_t* mask = lv.zoom_mask + (size_t)ck.bg * mask_words;
  const float scale2 = rsqrtf((float)kD) * kLog2e;
  const int row_end = ck.row_end;

  uint32_t qf[4][4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (gid < G) v = *reinterpret_cast<const uint4*>(q + ((size_t)b * Hq + (size_t)g * G + gid) * kD + (t4 + 4 * j) * 8);
    qf[j][0] = v.x; qf[j][1] = v.y; qf[j][2] = v.z; qf[j][3] = v.w;
  }
  float m_run = -INFINITY, l_run = 0.f;
  // acc[s][w][2o + c] = O[head 2*t4 + c][dim 64s + 8gid + 2w + o]
  float acc[2][4][4];
#pragma unroll
  for (int s = 0; s < 2; ++s)
#pragma unroll
    for (int w = 0; w < 4; ++w) { acc[s][w][0] = 0.f; acc[s][w][1] = 0.f; acc[s][w][2] = 0.f; acc[s][w][3] = 0.f; }

  const int ntiles = (row_end - ck.row_begin + 15) >> 4;
  uint4 kf[2][4], vf[4][2];
  auto load_k = [&](int t) {
    const int r0 = ck.row_begin + t * 16;
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
      const int row = min(r0 + 8 * nt + gid, row_end - 1);
      const uint8_t* p = Kb + (size_t)row * (kD * 2) + t4 * 16;
#pragma unroll
      for (int j = 0; j < 4; ++j) kf[nt][j] = ldg16(p + j * 64);
    }
  };
  auto load_v = [&](int t) {
    const int r0 = ck.row_begin + t * 16;
#pragma unroll
    for (int rr = 0; rr < 4; ++rr) {
      const int row = min(r0 + 2 * t4 + (rr & 1) + 8 * (rr >> 1), row_end - 1);
      const uint8_t* p = Vb + (size_t)row * (kD * 2) + gid * 16;
      vf[rr][0] = ldg16(p);
      vf[rr][1] = ldg16(p + 128);
    }
  };
  if (warp < ntiles) { load_k(warp); load_v(warp); }
  for (int t = warp; t < ntiles; t += NW) {
    const int r0 = ck.row_begin + t * 16;
    // S = Q K^T for 2 n-tiles of 8 tokens
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
    const bool more = (t + NW) < ntiles;
    if (more) load_k(t + NW);
    // logits in the base-2 domain with the entry bias (0 for pool tokens, ln|S| for coarse entries,
    // -inf for expanded spans and for rows past the chunk)
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
            bias = (mask[s >> 5] & (1u << (s & 31))) ? -INFINITY : cv.ln_len[span0 + s] * kLog2e;
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
      const float ca = __shfl_sync(0xffffffffu, corr, 8 * t4);       // head 2*t4   (lane gid = 2*t4, t4 = 0)
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
    // O^T += V^T P^T over 8 m-tiles of 16 dims
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
    if (more) load_v(t + NW);
  }
  // warp result -> shared memory
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
  cta_merge_store<G, NW>(sm_o, sm_ml, partials + (size_t)blockIdx.x * G * kPartStride);
}

// ---------------------------------------------------------------------------------------------
// Stage 2: one warp per expanded span, kStage2SpansPerCta warps per CTA
// ---------------------------------------------------------------------------------------------
template <int G>
__global__ void __launch_bounds__(kStage2SpansPerCta * 32)
stage2_mma_kernel(CsrView cv, LayerView lv, const int32_t* __restrict__ count, const __nv_bfloat16* __restrict__ q,
                  int Hq, int k_cap, int ways, int spans_cap, int64_t slot_bytes, float* __restrict__ partials) {
  constexpr int NW = kStage2SpansPerCta;
  __shared__ float sm_o[NW * G * kD];
  __shared__ float sm_ml[NW * G * 2];
  const int p = blockIdx.x, g = blockIdx.y, b = blockIdx.z, Hkv = gridDim.y, P2 = gridDim.x;
  const int bg = b * Hkv + g;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int gid = lane >> 2, t4 = lane & 3;
  const int cnt = min(count[bg], k_cap);
  const int j = p * NW + warp;
  const int id = (j < cnt) ? lv.item_span[(size_t)bg * k_cap + j] : -1;
  float m_run = -INFINITY, l_run = 0.f;
  float of[16][4];
#pragma unroll
  for (int n = 0; n < 16; ++n) { of[n][0] = of[n][1] = of[n][2] = of[n][3] = 0.f; }
  if (id >= 0) {                                       // warp-uniform
    const int way = (int)(lv.items[(size_t)bg * k_cap + j] & 0x7FFFFFFFu);
    const int gs = cv.seq_span_off[b] + id;
    const int rr = lv.dir_rank[(size_t)g * spans_cap + gs];
    const int len = cv.span_len[gs];
    const BlobDims bd = blob_dims(2, len, rr & 0xff, (rr >> 8) & 0xff);
    const uint8_t* blob = lv.slots + ((size_t)bg * ways + way) * slot_bytes;
    const float* sK = (const float*)(blob + bd.off_sk);
    const float* sV = (const float*)(blob + bd.off_sv);
    const uint8_t* VtK = blob + bd.off_vtk;
    const uint8_t* VV = blob + bd.off_vv;
    const uint8_t* UK = blob + bd.off_uk;
    const uint8_t* UVt = blob + bd.off_uvt;
    const int nks = (bd.rkp + 15) >> 4, nvs = (bd.rvp + 15) >> 4;     // k-steps over the key / value rank
    const float scale2 = rsqrtf((float)kD) * kLog2e;

    uint32_t qf[4][4];
#pragma unroll
    for (int jj = 0; jj < 4; ++jj) {
      uint4 v = make_uint4(0u, 0u, 0u, 0u);
      if (gid < G) v = *reinterpret_cast<const uint4*>(q + ((size_t)b * Hq + (size_t)g * G + gid) * kD + (t4 + 4 * jj) * 8);
      qf[jj][0] = v.x; qf[jj][1] = v.y; qf[jj][2] = v.z; qf[jj][3] = v.w;
    }
    // 1. c = sigma_K o (Vt_K q): rows of Vt_K play the role of tokens
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
          // rows past the padded rank do not exist: feed zeros (the mma itself is warp-wide)
          const bool have = irow < bd.rkp;
          const uint8_t* prow = VtK + (size_t)(have ? irow : 0) * (kD * 2) + t4 * 16;
#pragma unroll
          for (int jj = 0; jj < 4; ++jj) {
            uint4 kv = make_uint4(0u, 0u, 0u, 0u);
            if (have) kv = ldg16(prow + jj * 64);
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
    // 2. token groups of 16
    float yf[8][4];
#pragma unroll
    for (int n = 0; n < 8; ++n) { yf[n][0] = yf[n][1] = yf[n][2] = yf[n][3] = 0.f; }
    const int ngrp = bd.lenp >> 4;
    for (int grp = 0; grp < ngrp; ++grp) {
      float sacc[2][4];
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        sacc[u][0] = sacc[u][1] = sacc[u][2] = sacc[u][3] = 0.f;
        const int tok = 16 * grp + pi_index(u, gid);
        const uint8_t* prow = UK + (size_t)tok * (bd.rkp * 2) + t4 * 8;
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) {
          if (ks < nks) {
            uint2 bv = make_uint2(0u, 0u);
            if (16 * ks + 4 * t4 < bd.rkp) bv = ldg8(prow + ks * 32);
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
        for (int e = 0; e < 2; ++e) z[u][e] = (16 * grp + 4 * t4 + 2 * u + e < len) ? sacc[u][e] : -INFINITY;
      const float mx = quad_max(fmaxf(fmaxf(z[0][0], z[0][1]), fmaxf(z[1][0], z[1][1])));
      const float m_new = fmaxf(m_run, mx);
      const float m_safe = (m_new == -INFINITY) ? 0.f : m_new;
      if (__any_sync(0xffffffffu, m_new > m_run)) {
        const float corr = exp2f(m_run - m_safe);
        l_run *= corr;
#pragma unroll
        for (int n = 0; n < 8; ++n) { yf[n][0] *= corr; yf[n][1] *= corr; }
      }
      m_run = m_new;
      const float p00 = exp2f(z[0][0] - m_safe), p01 = exp2f(z[0][1] - m_safe);
      const float p10 = exp2f(z[1][0] - m_safe), p11 = exp2f(z[1][1] - m_safe);
      l_run += (p00 + p01) + (p10 + p11);
      uint32_t a0h, a0l, a2h, a2l;
      split_bf16(p00, p01, a0h, a0l);     // tokens 4*t4 + {0,1}  <-> k = 2*t4 + e
      split_bf16(p10, p11, a2h, a2l);     // tokens 4*t4 + {2,3}  <-> k = 8 + 2*t4 + e
      // y += P U_V : B[k = token][n = i] read from the transposed factor UVt[i][token]
#pragma unroll
      for (int n = 0; n < 8; ++n) {
        if (n < 2 * nvs) {
          const int irow = pi_index(n, gid);
          uint2 bv = make_uint2(0u, 0u);
          if (irow < bd.rvp) bv = ldg8(UVt + ((size_t)irow * bd.lenp + 16 * grp + 4 * t4) * 2);
          mma16816(yf[n], a0h, a2h, bv.x, bv.y);
          mma16816(yf[n], a0l, a2l, bv.x, bv.y);
        }
      }
    }
    // 3. o = (sigma_V o y) V_V^T ; yf[n][e] is head gid, rank index 16(n>>1) + 4*t4 + 2(n&1) + e
    uint32_t yh[4][2], yl[4][2];
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        yh[ks][u] = yl[ks][u] = 0u;
        if (ks < nvs) {
          const int i0 = 16 * ks + 4 * t4 + 2 * u;
          const float s0 = (i0 < bd.rvp) ? sV[i0] : 0.f;
          const float s1 = (i0 + 1 < bd.rvp) ? sV[i0 + 1] : 0.f;
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
          if (16 * ks + 4 * t4 < bd.rvp) bv = ldg8(prow + ks * 32);
          mma16816(of[nd], yh[ks][0], yh[ks][1], bv.x, bv.y);
          mma16816(of[nd], yl[ks][0], yl[ks][1], bv.x, bv.y);
        }
      }
    }
    l_run = quad_sum(l_run);
  }
  // of[nd][c] is head gid, dimension 8*nd + 2*t4 + c
  if (gid < G) {
    if (t4 == 0) { sm_ml[(warp * G + gid) * 2] = m_run; sm_ml[(warp * G + gid) * 2 + 1] = l_run; }
    float* o = sm_o + (warp * G + gid) * kD;
#pragma unroll
    for (int nd = 0; nd < 16; ++nd) { o[8 * nd + 2 * t4] = of[nd][0]; o[8 * nd + 2 * t4 + 1] = of[nd][1]; }
  }
  cta_merge_store<G, NW>(sm_o, sm_ml, partials + ((size_t)bg * P2 + p) * G * kPartStride);
}

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
bool have_mma_kernels() { return true; }

constexpr int kS1Warps = 4;

cudaError_t launch_stage1_mma(sekv_handle* h, int layer, const void* q, cudaStream_t s) {
  const sekv_config& c = h->cfg;
  if (h->n_chunks == 0) return cudaSuccess;
  CsrView cv = csr_view(h);
  LayerView lv = layer_view(h, layer);
  const Chunk* chunks = (const Chunk*)ws(h, h->F.off_chunks);
  float* partials = (float*)ws(h, h->F.off_partials1);
  const size_t ehs = (size_t)h->lay.rows_cap * kD;
#define SEKV_S1M(GG)                                                                                              \
  case GG:                                                                                                        \
    stage1_mma_kernel<GG, kS1Warps><<<h->n_chunks, kS1Warps * 32, 0, s>>>(                                        \
        cv, lv, chunks, (const __nv_bfloat16*)q, c.n_q_heads, c.n_kv_heads, ehs, h->mask_words, partials);        \
    break;
  switch (h->G) {
    SEKV_S1M(1) SEKV_S1M(2) SEKV_S1M(3) SEKV_S1M(4) SEKV_S1M(5) SEKV_S1M(6) SEKV_S1M(7) SEKV_S1M(8)
    default: return cudaErrorInvalidValue;
  }
#undef SEKV_S1M
  h->launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_stage2_mma(sekv_handle* h, int layer, const void* q, const int32_t* count, cudaStream_t s) {
  const sekv_config& c = h->cfg;
  CsrView cv = csr_view(h);
  LayerView lv = layer_view(h, layer);
  float* partials = (float*)ws(h, h->F.off_partials2);
  dim3 grid(h->P2, c.n_kv_heads, h->n_seqs);
#define SEKV_S2M(GG)                                                                                              \
  case GG:                                                                                                        \
    stage2_mma_kernel<GG><<<grid, kStage2SpansPerCta * 32, 0, s>>>(cv, lv, count, (const __nv_bfloat16*)q,        \
                                                                   c.n_q_heads, c.k_cap, c.cache_ways,            \
                                                                   (int)h->lay.spans_cap, h->lay.slot_bytes,      \
                                                                   partials);                                     \
    break;
  switch (h->G) {
    SEKV_S2M(1) SEKV_S2M(2) SEKV_S2M(3) SEKV_S2M(4) SEKV_S2M(5) SEKV_S2M(6) SEKV_S2M(7) SEKV_S2M(8)
    default: return cudaErrorInvalidValue;
  }
#undef SEKV_S2M
  h->launches += 1;
  return cudaGetLastError();
}

int stage1_mma_occupancy(int G) {
  int n = 0;
#define SEKV_OCC(GG) case GG: cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, stage1_mma_kernel<GG, kS1Warps>, kS1Warps * 32, 0); break;
  switch (G) { SEKV_OCC(1) SEKV_OCC(2) SEKV_OCC(3) SEKV_OCC(4) SEKV_OCC(5) SEKV_OCC(6) SEKV_OCC(7) SEKV_OCC(8) default: break; }
#undef SEKV_OCC
  return n;
}

}  // namespace sekv
