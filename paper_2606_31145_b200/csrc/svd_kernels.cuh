// Truncated SVD of every span's K (or V) matrix, Eq. 6 of PAPER.md, for the dense build mode.
// One CTA per (span, kv head): one-sided (Hestenes) Jacobi in shared memory, fp32.
//
// The |S| x 128 span matrix X is viewed as `nvec` vectors of length `vlen`, whichever side is smaller:
//   |S| >= 128: the 128 columns of X (vectors over tokens).   After convergence vec_j = sigma_j u_j.
//   |S| <  128: the |S| rows of X (vectors over dimensions).   After convergence vec_j = sigma_j v_j.
// Plane rotations orthogonalise the vectors; their norms are the singular values; the other side's
// singular vectors follow from X (re-read from global memory): v_j = X^T u_j / sigma_j, u_j = X v_j / sigma_j.
// Output layout = the prefactored build input: U rows token-indexed [tok][r], S [r], Vt [r][128];
// U and Vt are rounded to the storage dtype on write, sigma stays fp32 (reading #20).
// Sign and rotation ambiguities of singular vectors are immaterial: only products U S Vt are compared.
#pragma once

#include "sekv_internal.cuh"

namespace sekv {

constexpr int kSvdThreads = 256;
constexpr int kSvdMaxLen = 384;      // |S| x 128 fp32 must fit in shared memory (case |S| >= 128)
constexpr int kSvdMaxSweeps = 30;

template <typename ST>
__global__ void __launch_bounds__(kSvdThreads, 1)
span_svd_kernel(CsrView cv, const ST* __restrict__ X, size_t head_stride, ST* __restrict__ tokU,
                float* __restrict__ S, ST* __restrict__ Vt, size_t tok_tot, int m_tot, int r) {
  extern __shared__ float sm[];
  __shared__ float sh_norm2[256];
  __shared__ int sh_slot[256];
  __shared__ int sh_changed;
  const int s = blockIdx.x, g = blockIdx.y, tid = threadIdx.x;
  const int lane = tid & 31, warp = tid >> 5, nwarps = kSvdThreads >> 5;
  const int len = cv.span_len[s];
  const int64_t tok0 = cv.span_tok_start[s];
  const ST* Xs = X + (size_t)g * head_stride + (size_t)tok0 * kD;
  const bool caseA = len >= kD;
  const int nvec = caseA ? kD : len;
  const int vlen = caseA ? len : kD;
  const int ldv = vlen | 1;
  const int npad = (nvec + 1) & ~1;       // even number of players; the extra one is a zero vector
  // load
  for (int o = tid; o < len * kD; o += kSvdThreads) {
    const int t = o / kD, d = o % kD;
    const float v = StTraits<ST>::ld(Xs + o);
    if (caseA) sm[d * ldv + t] = v; else sm[t * ldv + d] = v;
  }
  if (npad > nvec) for (int i = tid; i < vlen; i += kSvdThreads) sm[nvec * ldv + i] = 0.f;
  __syncthreads();
  // sweeps
  for (int sweep = 0; sweep < kSvdMaxSweeps; ++sweep) {
    if (tid == 0) sh_changed = 0;
    __syncthreads();
    for (int round = 0; round < npad - 1; ++round) {
      for (int k = warp; k < npad / 2; k += nwarps) {
        // round-robin tournament: player npad-1 is fixed, the others rotate
        int p, q;
        if (k == 0) { p = npad - 1; q = round % (npad - 1); }
        else { p = (k + round) % (npad - 1); q = (npad - 1 - k + round) % (npad - 1); }
        float* vp = sm + p * ldv;
        float* vq = sm + q * ldv;
        float a = 0.f, b = 0.f, c = 0.f;
        for (int i = lane; i < vlen; i += 32) { const float x = vp[i], y = vq[i]; a = fmaf(x, x, a); b = fmaf(y, y, b); c = fmaf(x, y, c); }
        a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
        if (a > 0.f && b > 0.f && fabsf(c) > 1e-7f * sqrtf(a * b)) {
          const float zeta = (b - a) / (2.f * c);
          const float t = (zeta >= 0.f ? 1.f : -1.f) / (fabsf(zeta) + sqrtf(1.f + zeta * zeta));
          const float cs = rsqrtf(1.f + t * t), sn = cs * t;
          for (int i = lane; i < vlen; i += 32) {
            const float x = vp[i], y = vq[i];
            vp[i] = cs * x - sn * y;
            vq[i] = sn * x + cs * y;
          }
          if (lane == 0 && fabsf(c) > 1e-6f * sqrtf(a * b)) sh_changed = 1;
        }
      }
      __syncthreads();
    }
    const int ch = sh_changed;
    __syncthreads();
    if (!ch) break;
  }
  // singular values = vector norms; rank them (descending, ties to the lower index)
  for (int j = warp; j < nvec; j += nwarps) {
    float a = 0.f;
    for (int i = lane; i < vlen; i += 32) { const float x = sm[j * ldv + i]; a = fmaf(x, x, a); }
    a = warp_sum(a);
    if (lane == 0) sh_norm2[j] = a;
  }
  __syncthreads();
  if (tid < nvec) {
    const float mine = sh_norm2[tid];
    int rank = 0;
    for (int k = 0; k < nvec; ++k) { const float o = sh_norm2[k]; rank += (o > mine) || (o == mine && k < tid); }
    sh_slot[tid] = rank;
  }
  __syncthreads();
  const int keep = min(r, min(len, kD));
  ST* Uout = tokU + ((size_t)g * tok_tot + tok0) * r;
  float* Sout = S + ((size_t)g * m_tot + s) * r;
  ST* Vtout = Vt + ((size_t)g * m_tot + s) * r * kD;
  float max2 = 0.f;
  for (int k = 0; k < nvec; ++k) max2 = fmaxf(max2, sh_norm2[k]);
  for (int j = 0; j < nvec; ++j) {
    const int slot = sh_slot[j];
    if (slot >= keep) continue;                     // block-uniform
    const float n2 = sh_norm2[j];
    const bool ok = n2 > 1e-14f * max2 && n2 > 0.f;
    const float sig = ok ? sqrtf(n2) : 0.f;
    const float inv = ok ? 1.f / sig : 0.f, inv2 = ok ? 1.f / n2 : 0.f;
    const float* vj = sm + j * ldv;
    if (tid == 0) Sout[slot] = sig;
    if (caseA) {
      for (int t = tid; t < len; t += kSvdThreads) StTraits<ST>::st(Uout + (size_t)t * r + slot, vj[t] * inv);
      // v_j[d] = sum_t X[t][d] vec_j[t] / sigma^2
      if (tid < kD) {
        float acc = 0.f;
        for (int t = 0; t < len; ++t) acc = fmaf(StTraits<ST>::ld(Xs + (size_t)t * kD + tid), vj[t], acc);
        StTraits<ST>::st(Vtout + (size_t)slot * kD + tid, acc * inv2);
      }
    } else {
      if (tid < kD) StTraits<ST>::st(Vtout + (size_t)slot * kD + tid, vj[tid] * inv);
      // u_j[t] = X[t] . vec_j / sigma^2   (one warp per token)
      for (int t = warp; t < len; t += nwarps) {
        float acc = 0.f;
        for (int d = lane; d < kD; d += 32) acc = fmaf(StTraits<ST>::ld(Xs + (size_t)t * kD + d), vj[d], acc);
        acc = warp_sum(acc);
        if (lane == 0) StTraits<ST>::st(Uout + (size_t)t * r + slot, acc * inv2);
      }
    }
  }
}

template <typename ST>
cudaError_t launch_span_svd(sekv_handle* h, const CsrView& cv, const ST* X, ST* tokU, float* S, ST* Vt,
                            size_t tok_tot, int m_tot, int Hkv, int r) {
  int max_len = 0;
  for (int v : h->span_len_host) max_len = v > max_len ? v : max_len;
  if (max_len > kSvdMaxLen) return cudaErrorInvalidValue;
  size_t smem = 0;
  for (int v : h->span_len_host) {
    const int nvec = v >= kD ? kD : v, vlen = v >= kD ? v : kD;
    const size_t need = (size_t)(((nvec + 1) & ~1)) * (vlen | 1) * 4;
    smem = need > smem ? need : smem;
  }
  cudaError_t e = cudaFuncSetAttribute(span_svd_kernel<ST>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  dim3 grid(m_tot, Hkv);
  span_svd_kernel<ST><<<grid, kSvdThreads, smem, h->main>>>(cv, X, tok_tot * kD, tokU, S, Vt, tok_tot, m_tot, r);
  h->launches += 1;
  return cudaGetLastError();
}

}  // namespace sekv
