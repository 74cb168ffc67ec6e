// a0: prefill-time construction kernels (sec. 3.1-3.2): segmentation from surprisal,
// full-resolution gather, surprisal-weighted coarse means and routing summaries, factor blobs.
// Setup path: correctness-grade, not tuned against a roofline.
#include <algorithm>
#include <cstdio>

#include "sekv_internal.cuh"
#include "svd_kernels.cuh"

namespace sekv {

// ---------------------------------------------------------------------------------------------
// Segmentation (Eq. 17 window)
// ---------------------------------------------------------------------------------------------
__device__ double block_sum_double(double v, double* sh) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if (lane == 0) sh[w] = v;
  __syncthreads();
  double t = 0.0;
  for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += sh[i];
  return t;
}

// thr[b] = mu + alpha * sigma, population sigma, two-pass in fp64 (reading #1)
__global__ void seg_threshold_kernel(const float* __restrict__ H, const int64_t* __restrict__ tok_off,
                                     double alpha, double* __restrict__ thr) {
  __shared__ double sh[32];
  const int b = blockIdx.x;
  const int64_t t0 = tok_off[b], t1 = tok_off[b + 1];
  const double n = (double)(t1 - t0);
  double s = 0.0;
  for (int64_t t = t0 + threadIdx.x; t < t1; t += blockDim.x) s += (double)H[t];
  const double mu = block_sum_double(s, sh) / n;
  double q = 0.0;
  for (int64_t t = t0 + threadIdx.x; t < t1; t += blockDim.x) { double d = (double)H[t] - mu; q += d * d; }
  const double var = block_sum_double(q, sh) / n;
  if (threadIdx.x == 0) thr[b] = mu + alpha * sqrt(var);
}

// flag: 1 = full resolution because boundary (H_t > thr, strict) or inside the local window
__global__ void seg_flag_kernel(const float* __restrict__ H, const int64_t* __restrict__ tok_off,
                                const double* __restrict__ thr, int window, uint8_t* __restrict__ flag,
                                uint8_t* __restrict__ flag2) {
  const int b = blockIdx.y;
  const int64_t t0 = tok_off[b], t1 = tok_off[b + 1];
  const double th = thr[b];
  for (int64_t t = t0 + blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < t1; t += (int64_t)gridDim.x * blockDim.x) {
    uint8_t f = ((double)H[t] > th) || (t >= t1 - window) ? 1 : 0;
    flag[t] = f;
    flag2[t] = f;
  }
}

// One thread per run start: measure the run; runs < l_min join the pool (flag2 = 2), others become
// spans (flag2 = 3 at the first token, run length in len_at).  err: 1 = run longer than max_span_len.
__global__ void seg_runs_kernel(const int64_t* __restrict__ tok_off, const uint8_t* __restrict__ flag,
                                uint8_t* __restrict__ flag2, int32_t* __restrict__ len_at, int l_min,
                                int max_span_len, int* __restrict__ err) {
  const int b = blockIdx.y;
  const int64_t t0 = tok_off[b], t1 = tok_off[b + 1];
  for (int64_t t = t0 + blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < t1; t += (int64_t)gridDim.x * blockDim.x) {
    if (flag[t] != 0) continue;
    if (t > t0 && flag[t - 1] == 0) continue;   // not the first token of its run
    int len = 0;
    int64_t u = t;
    while (u < t1 && flag[u] == 0 && len <= max_span_len) { ++u; ++len; }
    if (len < l_min) {
      for (int64_t v = t; v < t + len; ++v) flag2[v] = 2;
    } else if (len > max_span_len) {
      atomicExch(err, 1);
    } else {
      flag2[t] = 3;
      len_at[t] = len;
    }
  }
}

__global__ void seg_count_kernel(const int64_t* __restrict__ tok_off, const uint8_t* __restrict__ flag2,
                                 int32_t* __restrict__ counts /* [B][2] = pool, spans */) {
  __shared__ int sh[2];
  const int b = blockIdx.x;
  if (threadIdx.x < 2) sh[threadIdx.x] = 0;
  __syncthreads();
  int p = 0, s = 0;
  for (int64_t t = tok_off[b] + threadIdx.x; t < tok_off[b + 1]; t += blockDim.x) {
    uint8_t f = flag2[t];
    p += (f == 1 || f == 2);
    s += (f == 3);
  }
  atomicAdd(&sh[0], p);
  atomicAdd(&sh[1], s);
  __syncthreads();
  if (threadIdx.x < 2) counts[b * 2 + threadIdx.x] = sh[threadIdx.x];
}

// Ordered compaction: one CTA per sequence walks its tokens in chunks with a block-wide scan.
__global__ void seg_compact_kernel(const int64_t* __restrict__ tok_off, const uint8_t* __restrict__ flag2,
                                   const int32_t* __restrict__ len_at, const int32_t* __restrict__ seq_pool_off,
                                   const int32_t* __restrict__ seq_span_off, int64_t* __restrict__ pool_tok,
                                   int64_t* __restrict__ span_tok_start, int32_t* __restrict__ span_len,
                                   float* __restrict__ ln_len) {
  __shared__ int warp_p[32], warp_s[32];
  __shared__ int base_p, base_s;
  const int b = blockIdx.x;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  if (threadIdx.x == 0) { base_p = seq_pool_off[b]; base_s = seq_span_off[b]; }
  __syncthreads();
  const int64_t t0 = tok_off[b], t1 = tok_off[b + 1];
  for (int64_t c0 = t0; c0 < t1; c0 += blockDim.x) {
    const int64_t t = c0 + threadIdx.x;
    const uint8_t f = t < t1 ? flag2[t] : 0;
    const int ip = (f == 1 || f == 2), is = (f == 3);
    const unsigned bp = __ballot_sync(0xffffffffu, ip), bs = __ballot_sync(0xffffffffu, is);
    const unsigned lower = (1u << lane) - 1u;
    if (lane == 0) { warp_p[w] = __popc(bp); warp_s[w] = __popc(bs); }
    __syncthreads();
    int op = 0, os = 0, tp = 0, ts = 0;
    for (int i = 0; i < nw; ++i) {
      if (i < w) { op += warp_p[i]; os += warp_s[i]; }
      tp += warp_p[i]; ts += warp_s[i];
    }
    if (ip) pool_tok[base_p + op + __popc(bp & lower)] = t;
    if (is) {
      const int idx = base_s + os + __popc(bs & lower);
      const int len = len_at[t];
      span_tok_start[idx] = t;
      span_len[idx] = len;
      ln_len[idx] = logf((float)len);
    }
    __syncthreads();
    if (threadIdx.x == 0) { base_p += tp; base_s += ts; }
    __syncthreads();
  }
}

// The four scan kernels of the segmentation rule on caller-provided scratch (also used by sekv_build_sizes):
// thresholds, boundary / window flags, run lengths (spans vs short runs), per-sequence counts.
cudaError_t segment_scan(const float* H, int n_seqs, const int64_t* tok_off_dev, double alpha, int window, int l_min,
                         int max_span_len, uint8_t* flag, uint8_t* flag2, int32_t* len_at, double* thr,
                         int32_t* counts, int* err, cudaStream_t s) {
  cudaError_t e;
  if ((e = cudaMemsetAsync(err, 0, 4, s)) != cudaSuccess) return e;
  seg_threshold_kernel<<<n_seqs, 1024, 0, s>>>(H, tok_off_dev, alpha, thr);
  dim3 grid(64, n_seqs);
  seg_flag_kernel<<<grid, 256, 0, s>>>(H, tok_off_dev, thr, window, flag, flag2);
  seg_runs_kernel<<<grid, 256, 0, s>>>(tok_off_dev, flag, flag2, len_at, l_min, max_span_len, err);
  seg_count_kernel<<<n_seqs, 1024, 0, s>>>(tok_off_dev, flag2, counts);
  return cudaGetLastError();
}

cudaError_t launch_segment(sekv_handle* h, const float* H, int n_seqs, const int64_t* tok_off_host, int* m_out,
                           int* a_out, std::string* why) {
  const sekv_config& c = h->cfg;
  cudaStream_t s = h->main;
  cudaError_t e;
  CsrView cv = csr_view(h);
  uint8_t* flag = ws(h, h->F.off_seg_flag);
  uint8_t* flag2 = ws(h, h->F.off_seg_flag2);
  int32_t* len_at = (int32_t*)ws(h, h->F.off_seg_len);
  double* thr = (double*)ws(h, h->F.off_seg_misc);
  int32_t* counts = (int32_t*)(ws(h, h->F.off_seg_misc) + (size_t)c.max_seqs * 8);
  int* err = (int*)ws(h, h->F.off_err_flag);
  if ((e = cudaMemcpyAsync((void*)cv.seq_tok_off, tok_off_host, (size_t)(n_seqs + 1) * 8, cudaMemcpyHostToDevice, s)) != cudaSuccess) return e;
  if ((e = segment_scan(H, n_seqs, cv.seq_tok_off, (double)c.alpha, c.window, c.l_min, c.max_span_len, flag, flag2,
                        len_at, thr, counts, err, s)) != cudaSuccess) return e;
  h->launches += 4;
  std::vector<int32_t> cnt((size_t)n_seqs * 2);
  int herr = 0;
  if ((e = cudaMemcpyAsync(cnt.data(), counts, cnt.size() * 4, cudaMemcpyDeviceToHost, s)) != cudaSuccess) return e;
  if ((e = cudaMemcpyAsync(&herr, err, 4, cudaMemcpyDeviceToHost, s)) != cudaSuccess) return e;
  if ((e = cudaStreamSynchronize(s)) != cudaSuccess) return e;
  if (herr) { *why = "a span is longer than max_span_len"; return cudaSuccess; }
  std::vector<int32_t> row_off(n_seqs + 1, 0), span_off(n_seqs + 1, 0), pool_off(n_seqs + 1, 0), pool_cnt(n_seqs, 0);
  for (int b = 0; b < n_seqs; ++b) {
    a_out[b] = cnt[b * 2]; m_out[b] = cnt[b * 2 + 1];
    if (m_out[b] > SEKV_MAX_SPANS_PER_SEQ) { *why = "more than 8192 spans in one sequence"; return cudaSuccess; }
    pool_cnt[b] = a_out[b];
    pool_off[b + 1] = pool_off[b] + a_out[b];
    span_off[b + 1] = span_off[b] + m_out[b];
    row_off[b + 1] = row_off[b] + a_out[b] + m_out[b];
  }
  if (span_off[n_seqs] > c.max_spans_total) { *why = "span capacity (max_spans_total) exceeded"; return cudaSuccess; }
  if (pool_off[n_seqs] > c.max_full_total) { *why = "full-resolution capacity (max_full_total) exceeded"; return cudaSuccess; }
  // pool offsets travel in the (unused until now) tail of seg_misc
  int32_t* d_pool_off = counts + (size_t)c.max_seqs * 2;
  if ((e = cudaMemcpyAsync((void*)cv.seq_row_off, row_off.data(), row_off.size() * 4, cudaMemcpyHostToDevice, s)) != cudaSuccess) return e;
  if ((e = cudaMemcpyAsync((void*)cv.seq_span_off, span_off.data(), span_off.size() * 4, cudaMemcpyHostToDevice, s)) != cudaSuccess) return e;
  if ((e = cudaMemcpyAsync((void*)cv.seq_pool_cnt, pool_cnt.data(), pool_cnt.size() * 4, cudaMemcpyHostToDevice, s)) != cudaSuccess) return e;
  if ((e = cudaMemcpyAsync(d_pool_off, pool_off.data(), (size_t)n_seqs * 4, cudaMemcpyHostToDevice, s)) != cudaSuccess) return e;
  seg_compact_kernel<<<n_seqs, 1024, 0, s>>>(cv.seq_tok_off, flag2, len_at, d_pool_off, cv.seq_span_off,
                                             (int64_t*)cv.pool_tok, (int64_t*)cv.span_tok_start,
                                             (int32_t*)cv.span_len, (float*)cv.ln_len);
  h->launches += 1;
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  h->span_len_host.resize(span_off[n_seqs]);
  if (span_off[n_seqs] > 0)
    if ((e = cudaMemcpyAsync(h->span_len_host.data(), cv.span_len, (size_t)span_off[n_seqs] * 4, cudaMemcpyDeviceToHost, s)) != cudaSuccess) return e;
  return cudaStreamSynchronize(s);
}

// ---------------------------------------------------------------------------------------------
// Shared by both build modes
// ---------------------------------------------------------------------------------------------
// global row of (sequence of span s, kind) helpers: the sequence of a global span index
__device__ __forceinline__ int seq_of_span(const int32_t* seq_span_off, int B, int s) {
  int b = 0;
  while (b + 1 < B && seq_span_off[b + 1] <= s) ++b;
  return b;
}

// copy W of this layer into the arena
template <typename ST>
__global__ void copy_kernel(const ST* __restrict__ src, ST* __restrict__ dst, size_t n) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}

// full-resolution rows: ent[g][row_off_b + a] = src[g][src_row(a)]
//   dense mode:       src_row = pool_tok[pool index]  (token-indexed K/V, L55 "retained ... at full resolution")
//   prefactored mode: src_row = pool index            (compact Kfull/Vfull)
template <typename ST>
__global__ void gather_pool_kernel(const ST* __restrict__ srcK, const ST* __restrict__ srcV, size_t src_head_stride,
                                   const int64_t* __restrict__ pool_tok, int dense, CsrView cv, int B,
                                   ST* __restrict__ entK, ST* __restrict__ entV, size_t ent_head_stride) {
  const int g = blockIdx.y;
  // blockIdx.x walks global pool indices, 2 per block (64 threads each, 2 elements per thread)
  int pool_base = 0;
  for (int b = 0; b < B; ++b) {
    const int A = cv.seq_pool_cnt[b];
    for (int a = blockIdx.x * 2 + (threadIdx.x >> 6); a < A; a += gridDim.x * 2) {
      const int64_t srow = dense ? pool_tok[pool_base + a] : (int64_t)(pool_base + a);
      const size_t so = (size_t)g * src_head_stride + (size_t)srow * kD;
      const size_t dofs = (size_t)g * ent_head_stride + (size_t)(cv.seq_row_off[b] + a) * kD;
      const int d = (threadIdx.x & 63) * 2;
      entK[dofs + d] = srcK[so + d]; entK[dofs + d + 1] = srcK[so + d + 1];
      entV[dofs + d] = srcV[so + d]; entV[dofs + d + 1] = srcV[so + d + 1];
    }
    pool_base += A;
  }
}

__device__ float block_sum_float(float v, float* sh) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  v = warp_sum(v);
  __syncthreads();
  if (lane == 0) sh[w] = v;
  __syncthreads();
  float t = 0.f;
  for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += sh[i];
  return t;
}

// Coarse means and routing summaries of one (span, kv head): block of 128 threads.
//   w_t = H_t / sum H (Eq. 2; uniform if the sum is 0, reading #6)
//   k_bar = sum_t w_t K_t, v_bar = sum_t w_t V_t (L81)  -> entry rows after the sequence's pool rows
//   K_bar^(h) = normalize(W^(h) k_bar) for every query head of the group (Eq. 3, by linearity)
// MODE 0: K_t rows read from dense K/V.  MODE 1: K_t = tokU[t] diag(S) Vt, so
//   k_bar = ((w^T tokU) o S) Vt.
template <typename ST, int MODE>
__global__ void summary_kernel(const float* __restrict__ H, CsrView cv, int B, int G, int dp,
                               const ST* __restrict__ Kd, const ST* __restrict__ Vd, size_t dense_head_stride,
                               sekv_factors f, size_t tok_tot, int m_tot,
                               const ST* __restrict__ W, ST* __restrict__ entK, ST* __restrict__ entV,
                               size_t ent_head_stride, ST* __restrict__ route, size_t route_head_stride) {
  __shared__ float sh_red[32];
  __shared__ float sh_w[SEKV_MAX_SPAN_LEN];
  __shared__ float sh_a[2][SEKV_MAX_RANK];
  __shared__ float sh_kbar[kD];
  __shared__ float sh_p[SEKV_MAX_GROUP * SEKV_MAX_ROUTE_DIM];
  const int s = blockIdx.x, g = blockIdx.y, tid = threadIdx.x;
  const int b = seq_of_span(cv.seq_span_off, B, s);
  const int len = cv.span_len[s];
  const int64_t tok0 = cv.span_tok_start[s];
  // weights
  float hs = 0.f;
  for (int t = tid; t < len; t += blockDim.x) { float v = H[tok0 + t]; sh_w[t] = v; hs += v; }
  const float tot = block_sum_float(hs, sh_red);
  __syncthreads();
  for (int t = tid; t < len; t += blockDim.x) sh_w[t] = (tot == 0.f) ? 1.f / (float)len : sh_w[t] / tot;
  __syncthreads();
  float kbar = 0.f, vbar = 0.f;   // thread tid owns dimension tid
  if (MODE == 0) {
    const ST* kp = Kd + (size_t)g * dense_head_stride + (size_t)tok0 * kD + tid;
    const ST* vp = Vd + (size_t)g * dense_head_stride + (size_t)tok0 * kD + tid;
    for (int t = 0; t < len; ++t) {
      kbar = fmaf(sh_w[t], StTraits<ST>::ld(kp + (size_t)t * kD), kbar);
      vbar = fmaf(sh_w[t], StTraits<ST>::ld(vp + (size_t)t * kD), vbar);
    }
  } else {
    const int r = f.rank_in;
    const ST* uk = (const ST*)f.tokUK + ((size_t)g * tok_tot + tok0) * r;
    const ST* uv = (const ST*)f.tokUV + ((size_t)g * tok_tot + tok0) * r;
    // a[i] = S_i * sum_t w_t U[t][i]   (threads 0..r-1 for K, 64..64+r-1 for V)
    const int side = tid >> 6, i = tid & 63;
    if (i < r) {
      const ST* u = side ? uv : uk;
      float acc = 0.f;
      for (int t = 0; t < len; ++t) acc = fmaf(sh_w[t], StTraits<ST>::ld(u + (size_t)t * r + i), acc);
      const float* S = (side ? f.SV : f.SK) + ((size_t)g * m_tot + s) * r;
      sh_a[side][i] = acc * S[i];
    }
    __syncthreads();
    const ST* vtk = (const ST*)f.VtK + ((size_t)g * m_tot + s) * r * kD;
    const ST* vtv = (const ST*)f.VtV + ((size_t)g * m_tot + s) * r * kD;
    for (int j = 0; j < r; ++j) {
      kbar = fmaf(sh_a[0][j], StTraits<ST>::ld(vtk + (size_t)j * kD + tid), kbar);
      vbar = fmaf(sh_a[1][j], StTraits<ST>::ld(vtv + (size_t)j * kD + tid), vbar);
    }
  }
  const size_t row = (size_t)cv.seq_row_off[b] + cv.seq_pool_cnt[b] + (s - cv.seq_span_off[b]);
  StTraits<ST>::st(entK + (size_t)g * ent_head_stride + row * kD + tid, kbar);
  StTraits<ST>::st(entV + (size_t)g * ent_head_stride + row * kD + tid, vbar);
  sh_kbar[tid] = kbar;
  __syncthreads();
  // routing summaries: P[hl][j] = W[h][j] . k_bar
  for (int o = tid; o < G * dp; o += blockDim.x) {
    const int hl = o / dp, j = o % dp;
    const ST* wr = W + ((size_t)(g * G + hl) * dp + j) * kD;
    float acc = 0.f;
    for (int d = 0; d < kD; ++d) acc = fmaf(StTraits<ST>::ld(wr + d), sh_kbar[d], acc);
    sh_p[o] = acc;
  }
  __syncthreads();
  for (int hl = 0; hl < G; ++hl) {
    float v = tid < dp ? sh_p[hl * dp + tid] : 0.f;
    const float n2 = block_sum_float(v * v, sh_red);
    const float nrm = sqrtf(n2);
    if (tid < dp) {
      const float o = nrm > 0.f ? v / nrm : 0.f;
      StTraits<ST>::st(route + (size_t)(g * G + hl) * route_head_stride + (size_t)s * dp + tid, o);
    }
  }
}

// Pack one (span, kv head) factor blob into the pinned host arena (device-mapped writes).
// Source: token-indexed U rows [tok][r_in], S [r_in], Vt [r_in][128] (prefactored input, or the SVD
// workspace in dense mode, which uses the same intermediate layout).
template <typename ST>
__global__ void pack_blob_kernel(CsrView cv, sekv_factors f, size_t tok_tot, int m_tot,
                                 const int64_t* __restrict__ dir_off, const int32_t* __restrict__ dir_rank,
                                 int spans_cap, uint8_t* __restrict__ host_arena) {
  const int s = blockIdx.x, g = blockIdx.y, tid = threadIdx.x, nt = blockDim.x;
  const int len = cv.span_len[s];
  const int64_t tok0 = cv.span_tok_start[s];
  const int rr = dir_rank[(size_t)g * spans_cap + s];
  const int rk = rr & 0xff, rv = (rr >> 8) & 0xff;
  const BlobDims bd = blob_dims((int)sizeof(ST), len, rk, rv);
  uint8_t* blob = host_arena + dir_off[(size_t)g * spans_cap + s];
  const int r = f.rank_in;
  const float* SK = f.SK + ((size_t)g * m_tot + s) * r;
  const float* SV = f.SV + ((size_t)g * m_tot + s) * r;
  float* bsk = (float*)(blob + bd.off_sk);
  float* bsv = (float*)(blob + bd.off_sv);
  for (int i = tid; i < bd.rkp; i += nt) bsk[i] = i < rk ? SK[i] : 0.f;
  for (int i = tid; i < bd.rvp; i += nt) bsv[i] = i < rv ? SV[i] : 0.f;
  const ST zero = ST(0.f);
  // The loops run over the DESTINATION in address order (coalesced writes to the mapped host store) and invert
  // the fragment-order maps of blob_vtk_off / blob_vv_off / blob_uk_off / blob_uv_off (sekv_internal.cuh).
  const ST* vtk = (const ST*)f.VtK + ((size_t)g * m_tot + s) * r * kD;
  ST* bvtk = (ST*)(blob + bd.off_vtk);
  for (int o = tid; o < bd.rkp * kD; o += nt) {
    const int e8 = o & 7, lane = (o >> 3) & 31, blk = o >> 8;
    const int jj = blk & 3, u = (blk >> 2) & 1, ks = blk >> 3, gid = lane >> 2, t4 = lane & 3;
    const int i = 16 * ks + 4 * (gid >> 1) + 2 * u + (gid & 1), d = 32 * jj + 8 * t4 + e8;
    bvtk[o] = i < rk ? vtk[(size_t)i * kD + d] : zero;
  }
  const ST* vtv = (const ST*)f.VtV + ((size_t)g * m_tot + s) * r * kD;
  ST* bvv = (ST*)(blob + bd.off_vv);
  for (int o = tid; o < kD * bd.rvp; o += nt) {
    const int e = o & 1, reg = (o >> 1) & 3, lane = (o >> 3) & 31, blk = o >> 8;
    const int md = blk & 7, kv = blk >> 3, gid = lane >> 2, t4 = lane & 3, half = reg >> 1, hi = reg & 1;
    const int d = 16 * md + 8 * hi + gid, i = 16 * kv + 8 * half + 2 * t4 + e;
    bvv[o] = i < rv ? vtv[(size_t)i * kD + d] : zero;
  }
  const ST* uk = (const ST*)f.tokUK + ((size_t)g * tok_tot + tok0) * r;
  const ST* uv = (const ST*)f.tokUV + ((size_t)g * tok_tot + tok0) * r;
  const int per_chunk = kLenPad * (bd.rkp + bd.rvp);
  ST* bch = (ST*)(blob + bd.off_chunks);
  for (int o = tid; o < (bd.lenp / kLenPad) * per_chunk; o += nt) {
    const int c = o / per_chunk, w = o % per_chunk;
    const int r8 = w & 7, lane = (w >> 3) & 31, blk = w >> 8, gid = lane >> 2, t4 = lane & 3;
    ST v = zero;
    if (blk < bd.nks) {
      const int t = 16 * c + 8 * (r8 >> 2) + gid, i = 16 * blk + 4 * t4 + (r8 & 3);
      if (t < len && i < rk) v = uk[(size_t)t * r + i];
    } else {
      const int reg = r8 >> 1, half = reg >> 1, hi = reg & 1;
      const int t = 16 * c + 8 * half + 2 * t4 + (r8 & 1), i = 16 * (blk - bd.nks) + 8 * hi + gid;
      if (t < len && i < rv) v = uv[(size_t)t * r + i];
    }
    bch[o] = v;
  }
  // tail padding up to the 128-byte blob size
  const size_t used = bd.off_chunks + (size_t)(bd.lenp / kLenPad) * bd.chunk_bytes;
  for (size_t o = used + tid; o < bd.bytes; o += nt) blob[o] = 0;
}

template <typename ST>
static cudaError_t build_common(sekv_handle* h, int layer, const float* H, int mode, const ST* Kd, const ST* Vd,
                                const sekv_factors& f, const void* W) {
  const sekv_config& c = h->cfg;
  cudaStream_t s = h->main;
  CsrView cv = csr_view(h);
  LayerView lv = layer_view(h, layer);
  const int B = h->n_seqs, Hkv = c.n_kv_heads;
  const size_t ent_hs = (size_t)h->lay.rows_cap * kD;
  const size_t route_hs = (size_t)h->lay.spans_cap * c.route_dim;
  const size_t tok_tot = (size_t)h->tok_off[B];
  const size_t wn = (size_t)c.n_q_heads * c.route_dim * kD;
  copy_kernel<ST><<<64, 256, 0, s>>>((const ST*)W, (ST*)lv.W, wn);
  h->launches += 1;
  if (h->A_tot > 0) {
    dim3 grid(std::min(std::max(h->A_tot / 2, 1), 2048), Hkv);
    if (mode == 0)
      gather_pool_kernel<ST><<<grid, 128, 0, s>>>(Kd, Vd, tok_tot * kD, cv.pool_tok, 1, cv, B, (ST*)lv.ent_k, (ST*)lv.ent_v, ent_hs);
    else
      gather_pool_kernel<ST><<<grid, 128, 0, s>>>((const ST*)f.Kfull, (const ST*)f.Vfull, (size_t)h->A_tot * kD, cv.pool_tok, 0, cv, B, (ST*)lv.ent_k, (ST*)lv.ent_v, ent_hs);
    h->launches += 1;
  }
  if (h->m_tot > 0) {
    dim3 grid(h->m_tot, Hkv);
    if (mode == 0)
      summary_kernel<ST, 0><<<grid, 128, 0, s>>>(H, cv, B, h->G, c.route_dim, Kd, Vd, tok_tot * kD, f, tok_tot, h->m_tot,
                                                 (const ST*)lv.W, (ST*)lv.ent_k, (ST*)lv.ent_v, ent_hs, (ST*)lv.route, route_hs);
    else
      summary_kernel<ST, 1><<<grid, 128, 0, s>>>(H, cv, B, h->G, c.route_dim, nullptr, nullptr, 0, f, tok_tot, h->m_tot,
                                                 (const ST*)lv.W, (ST*)lv.ent_k, (ST*)lv.ent_v, ent_hs, (ST*)lv.route, route_hs);
    pack_blob_kernel<ST><<<grid, 256, 0, s>>>(cv, f, tok_tot, h->m_tot, lv.dir_off, lv.dir_rank, (int)h->lay.spans_cap, h->host_dev);
    h->launches += 2;
  }
  return cudaGetLastError();
}

cudaError_t launch_build_prefactored(sekv_handle* h, int layer, const float* H, const sekv_factors* f, const void* W) {
  if (h->cfg.dtype == SEKV_BF16) return build_common<__nv_bfloat16>(h, layer, H, 1, nullptr, nullptr, *f, W);
  return build_common<float>(h, layer, H, 1, nullptr, nullptr, *f, W);
}

// Dense mode: truncated SVD of every span's K and V (Eq. 6) into a temporary workspace that has the
// prefactored intermediate layout, then the common path (summaries from the dense rows).
template <typename ST>
static cudaError_t build_dense_t(sekv_handle* h, int layer, const float* H, const ST* K, const ST* V, const void* W,
                                 int rank_cap, std::string* why) {
  const sekv_config& c = h->cfg;
  const int B = h->n_seqs, Hkv = c.n_kv_heads, m = h->m_tot;
  const size_t tok_tot = (size_t)h->tok_off[B];
  const int r = rank_cap;
  // temporary workspace (setup path only): token-indexed U, S, Vt for K and V
  const size_t u_bytes = (size_t)Hkv * tok_tot * r * sizeof(ST);
  const size_t s_bytes = (size_t)Hkv * std::max(m, 1) * r * 4;
  const size_t vt_bytes = (size_t)Hkv * std::max(m, 1) * r * kD * sizeof(ST);
  uint8_t* tmp = nullptr;
  const size_t total = 2 * (round_up_sz(u_bytes, 256) + round_up_sz(s_bytes, 256) + round_up_sz(vt_bytes, 256));
  cudaError_t e = cudaMalloc(&tmp, total);
  if (e != cudaSuccess) { *why = "cudaMalloc of the SVD workspace failed"; cudaGetLastError(); return cudaSuccess; }
  size_t o = 0;
  auto take = [&](size_t n) { uint8_t* p = tmp + o; o += round_up_sz(n, 256); return p; };
  sekv_factors f;
  memset(&f, 0, sizeof(f));
  f.rank_in = r;
  f.tokUK = take(u_bytes); f.SK = (const float*)take(s_bytes); f.VtK = take(vt_bytes);
  f.tokUV = take(u_bytes); f.SV = (const float*)take(s_bytes); f.VtV = take(vt_bytes);
  f.m_tot = m; f.a_tot = h->A_tot;
  e = cudaMemsetAsync(tmp, 0, total, h->main);
  if (e == cudaSuccess && m > 0) {
    CsrView cv = csr_view(h);
    e = launch_span_svd<ST>(h, cv, K, (ST*)f.tokUK, (float*)f.SK, (ST*)f.VtK, tok_tot, m, Hkv, r);
    if (e == cudaSuccess) e = launch_span_svd<ST>(h, cv, V, (ST*)f.tokUV, (float*)f.SV, (ST*)f.VtV, tok_tot, m, Hkv, r);
  }
  if (e == cudaSuccess) e = build_common<ST>(h, layer, H, 0, K, V, f, W);
  cudaError_t e2 = cudaStreamSynchronize(h->main);
  cudaFree(tmp);
  return e != cudaSuccess ? e : e2;
}

cudaError_t launch_build_dense(sekv_handle* h, int layer, const float* H, const void* K, const void* V, const void* W,
                               int rank_cap, std::string* why) {
  if (h->cfg.dtype == SEKV_BF16)
    return build_dense_t<__nv_bfloat16>(h, layer, H, (const __nv_bfloat16*)K, (const __nv_bfloat16*)V, W, rank_cap, why);
  return build_dense_t<float>(h, layer, H, (const float*)K, (const float*)V, W, rank_cap, why);
}

}  // namespace sekv

// ---------------------------------------------------------------------------------------------
// sekv_segment_counts_static (include/sekv.h): the four scan kernels of the segmentation rule on scratch that
// is NOT allocated: a file-scope device array.  In host code `g_static_scratch` is only a stand-in for the
// symbol, not a device address; the address a kernel can use comes from cudaGetSymbolAddress, looked up once
// per device (with that device current) and kept in g_static_ptr.
// ---------------------------------------------------------------------------------------------
namespace {

constexpr size_t kStOffFlag = 0;                                                   // uint8 [tokens]
constexpr size_t kStOffFlag2 = kStOffFlag + (size_t)SEKV_STATIC_MAX_TOKENS;         // uint8 [tokens]
constexpr size_t kStOffLen = kStOffFlag2 + (size_t)SEKV_STATIC_MAX_TOKENS;          // int32 [tokens]
constexpr size_t kStOffTok = kStOffLen + (size_t)SEKV_STATIC_MAX_TOKENS * 4;        // int64 [seqs + 1]
constexpr size_t kStOffThr = kStOffTok + (((size_t)SEKV_STATIC_MAX_SEQS + 1) * 8 + 255) / 256 * 256;   // double [seqs]
constexpr size_t kStBytes = kStOffThr + (size_t)SEKV_STATIC_MAX_SEQS * 8;
static_assert(kStOffLen % 256 == 0 && kStOffTok % 256 == 0 && kStOffThr % 256 == 0, "scratch alignment");

static __device__ __align__(256) uint8_t g_static_scratch[kStBytes];

constexpr int kStMaxDevices = 64;
uint8_t* g_static_ptr[kStMaxDevices];              // device address of g_static_scratch per device (null: not looked up)
thread_local const char* g_static_err = "";

sekv_status static_fail(sekv_status st, const char* msg) { g_static_err = msg; return st; }

}  // namespace

extern "C" const char* sekv_static_last_error(void) { return g_static_err; }

extern "C" sekv_status sekv_segment_counts_static(const sekv_config* cfg, int32_t n_seqs, const int64_t* seq_tok_off,
                                                  const float* H, int32_t* counts, int32_t* too_long, void* stream) {
  using namespace sekv;
  if (!cfg || !seq_tok_off || !H || !counts || !too_long) return static_fail(SEKV_INVALID_ARG, "NULL argument");
  if (n_seqs < 1) return static_fail(SEKV_INVALID_ARG, "n_seqs < 1");
  if (cfg->l_min < 1 || cfg->window < 0 || !(cfg->alpha == cfg->alpha))
    return static_fail(SEKV_INVALID_ARG, "bad cfg (l_min < 1, window < 0 or alpha is NaN)");
  if (n_seqs > SEKV_STATIC_MAX_SEQS)
    return static_fail(SEKV_UNSUPPORTED, "n_seqs exceeds SEKV_STATIC_MAX_SEQS (1024): use sekv_build_sizes");
  if (seq_tok_off[0] != 0) return static_fail(SEKV_INVALID_ARG, "seq_tok_off[0] != 0");
  for (int b = 0; b < n_seqs; ++b)
    if (seq_tok_off[b + 1] <= seq_tok_off[b]) return static_fail(SEKV_INVALID_ARG, "seq_tok_off is not increasing");
  if (seq_tok_off[n_seqs] > (int64_t)SEKV_STATIC_MAX_TOKENS)
    return static_fail(SEKV_UNSUPPORTED, "token count exceeds SEKV_STATIC_MAX_TOKENS (1048576): use sekv_build_sizes");
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return static_fail(SEKV_CUDA, "cudaGetDevice failed"); }
  if (dev < 0 || dev >= kStMaxDevices) return static_fail(SEKV_UNSUPPORTED, "device ordinal >= 64");
  uint8_t* base = g_static_ptr[dev];
  if (base == nullptr) {                    // first call on this device (racing threads store the same value)
    void* p = nullptr;
    const cudaError_t ge = cudaGetSymbolAddress(&p, g_static_scratch);
    if (ge != cudaSuccess || p == nullptr) {
      cudaGetLastError();
      return static_fail(SEKV_CUDA, "cudaGetSymbolAddress of the static scratch failed");
    }
    base = g_static_ptr[dev] = (uint8_t*)p;
  }
  cudaStream_t s = (cudaStream_t)stream;
  // (pageable host memory is staged before cudaMemcpyAsync returns: the caller's array may be reused at once)
  cudaError_t e = cudaMemcpyAsync(base + kStOffTok, seq_tok_off, (size_t)(n_seqs + 1) * 8, cudaMemcpyHostToDevice, s);
  // segment_scan clears *too_long itself; every other scratch byte a kernel reads was written by an earlier kernel
  // of this call (flags for every token, run lengths at the span starts that are read back), so the previous
  // call's contents are never seen
  if (e == cudaSuccess)
    e = segment_scan(H, n_seqs, (const int64_t*)(base + kStOffTok), (double)cfg->alpha, cfg->window, cfg->l_min,
                     SEKV_MAX_SPAN_LEN, base + kStOffFlag, base + kStOffFlag2, (int32_t*)(base + kStOffLen),
                     (double*)(base + kStOffThr), counts, too_long, s);
  if (e != cudaSuccess) { cudaGetLastError(); return static_fail(SEKV_CUDA, cudaGetErrorString(e)); }
  return SEKV_OK;
}
