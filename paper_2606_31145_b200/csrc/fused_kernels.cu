// The bf16 hot path: ONE persistent kernel per layer-step that runs a1-a7 (Eq. 4, 5, 9, L123,
// L119-121, Eq. 8).  One CTA per SM; every WARP is an independent worker with a private shared-memory
// region and pulls work items from two dependency-ordered queues (first item static, then atomic claims
// two items ahead so neither the claim nor the descriptor load is on the warp's critical path):
//
//   latency queue (even warps start here)
//     QPROJ   (b, h)              q' = W q (Eq. 4) on the tensor cores; published through a sentinel, no flag
//     ROUTE   (b, g, 64 spans)    x = q'.K_bar/sqrt(d') + ln|S|, alpha = sig(x) (Eq. 5), X = max over the group
//                                 (GQA), ordered 32-bit keys -> global
//     SELECT  (b, g)              top-k (Eq. 9, cap L123) by a 4-pass radix select on the keys, ties to the lower
//                                 span id, sorted ids; then the residency plan of the device factor cache (LRU),
//                                 zoom bit-mask, one descriptor per expanded span
//   main queue
//     POOL    (b, g, row range)   online-softmax partial over full-resolution tokens (no dependency): K/V rows
//                                 stream through a 3-stage cp.async ring (XOR-swizzled, bank-conflict free)
//     ZOOM    (b, g, plan items)  expanded spans through the factored form; the span's factor blob moves by ONE
//                                 1-D bulk async copy (TMA engine) into the warp's region -- from its cache slot
//                                 on a hit, straight from the pinned-host store over PCIe on a demand miss (and is
//                                 then written to the slot)
//     COARSE  (b, g, row range)   partial over the unexpanded coarse entries (+ln|S|); needs the zoom mask
//     COMBINE (b, h)              log-sum-exp merge of the head's partials -> output (a7)
//
// Waiting items only ever wait on items earlier in their queue (or in the latency queue), claims are in
// queue order and the grid is resident (one CTA per SM), so the wait graph is acyclic.
//
// Tensor cores: G <= 8 query heads per kv head is far below a tcgen05 tile and the path is HBM-bound, so
// the heads are the (padded) 16 rows of warp-level mma.sync.m16n8k16 tiles.
#include <algorithm>

#include "mma_common.cuh"

namespace sekv {

namespace {

constexpr int kStages = 3;                 // ring stages of a rows item (16 rows of K + 16 rows of V each)
constexpr int kStageBytes = 2 * 16 * kD * 2;

// Monotone map float -> uint32 (larger float => larger key); key 0 is free to mean "not eligible".
__device__ __forceinline__ uint32_t order_key(float x) {
  const uint32_t u = __float_as_uint(x);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

__device__ __forceinline__ void cp_async16(void* dst_smem, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ void red_add_release(int32_t* p, int v) {
  asm volatile("red.release.gpu.global.add.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ int warp_sum_i(int v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
// exclusive prefix sum over the warp
__device__ __forceinline__ int warp_excl_scan(int v, int lane) {
  int s = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int t = __shfl_up_sync(0xffffffffu, s, o);
    if (lane >= o) s += t;
  }
  return s - v;
}

// per-group counters inside P.ctrs
__device__ __forceinline__ int32_t* grp_ctr(const FusedParams& P, int bg, int which) { return P.ctrs + 4 + 4 * bg + which; }
enum { C_EARLY = 0, C_ROUTE = 1, C_ATTN = 2, C_PLAN = 3 };   // C_EARLY: POOL + COARSE items done

// spin (lane 0) until the counter reaches `target`
// (relaxed polls -- an acquire load would flush L1 on every poll -- then one acquire fence)
__device__ __forceinline__ void wait_ctr(const int32_t* c, int target, int lane, unsigned long long* t_mid = nullptr) {
  if (lane == 0) {
    int v;
    for (;;) {
      asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(c) : "memory");
      if (v >= target) break;
      __nanosleep(64);
    }
    asm volatile("fence.acq_rel.gpu;" ::: "memory");
    if (t_mid) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(*t_mid));
  }
  __syncwarp();
}
// trace mark k (1..3) of the current item (lane 0; tm = null when tracing is off)
__device__ __forceinline__ void mark(unsigned long long* tm, int k, int lane) {
  if (tm && lane == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tm[k]));
}
// every lane's earlier global writes happen-before the counter increment: __syncwarp orders them before
// lane 0's release (cumulativity), so no separate fence is needed
__device__ __forceinline__ void signal_ctr(int32_t* c, int lane) {
  __syncwarp();
  if (lane == 0) red_add_release(c, 1);
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

constexpr uint32_t kQpSentinel = 0xFFFFFFFFu;   // never produced by the tensor cores (their NaN is 0x7FFFFFFF)

// ---------------------------------------------------------------------------------------------------
// a1 (Eq. 4): q'_h = W_h q_h for one query head on the tensor cores: the rows of W_h are the M dimension
// (16 per tile), the group's queries are the 8 columns, column hl of the result is q'_hl.  All loads of
// W_h (dp x 128 bf16) are in flight at once.  The result is published without a flag: the buffer holds a
// sentinel bit pattern until the value arrives, and ROUTE items poll the words they need.
// ---------------------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ void qproj_item(const FusedParams& P, const Item& I, int lane) {
  const int bg = I.bg, b = bg / P.Hkv, g = bg % P.Hkv, dp = P.dp, hl = I.a;
  const int gid = lane >> 2, t4 = lane & 3;
  uint32_t qf[4][4];
  load_q_frags(P.q + ((size_t)b * P.Hq + (size_t)g * G) * kD, G, gid, t4, qf);
  const uint8_t* Wh = (const uint8_t*)P.lv.W + (size_t)(g * G + hl) * dp * (kD * 2) + t4 * 16;
  float* dst = P.qp + ((size_t)bg * G + hl) * dp;
#pragma unroll 1
  for (int j0 = 0; j0 < dp; j0 += 32) {
    uint4 w[2][2][4];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
      for (int hf = 0; hf < 2; ++hf) {
        const int row = j0 + 16 * mt + 8 * hf + gid;
#pragma unroll
        for (int jj = 0; jj < 4; ++jj)
          w[mt][hf][jj] = row < dp ? ldg16(Wh + (size_t)row * (kD * 2) + jj * 64) : make_uint4(0u, 0u, 0u, 0u);
      }
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
      float c[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int jj = 0; jj < 4; ++jj) {
        mma16816_full(c, w[mt][0][jj].x, w[mt][1][jj].x, w[mt][0][jj].y, w[mt][1][jj].y, qf[jj][0], qf[jj][1]);
        mma16816_full(c, w[mt][0][jj].z, w[mt][1][jj].z, w[mt][0][jj].w, w[mt][1][jj].w, qf[jj][2], qf[jj][3]);
      }
      if (t4 == (hl >> 1)) {                                     // this lane holds column hl of the tile
        const int r = j0 + 16 * mt + gid;
        if (r < dp) dst[r] = (hl & 1) ? c[1] : c[0];
        if (r + 8 < dp) dst[r + 8] = (hl & 1) ? c[3] : c[2];
      }
    }
  }
}

// poll four consecutive words of q' until none is the sentinel
__device__ __forceinline__ float4 poll_qp4(const float* p) {
  uint4 v;
  for (;;) {
    asm volatile("ld.relaxed.gpu.global.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    if (v.x != kQpSentinel && v.y != kQpSentinel && v.z != kQpSentinel && v.w != kQpSentinel) break;
    __nanosleep(64);
  }
  return make_float4(__uint_as_float(v.x), __uint_as_float(v.y), __uint_as_float(v.z), __uint_as_float(v.w));
}

// ---------------------------------------------------------------------------------------------------
// a2 + GQA reduce of a3 (Eq. 5, Eq. 9): spans [I.a, I.b) of (b, g).  The G x nsp rows of the routing table
// (dp bf16 each) are staged into the warp's region by 16-byte cp.async copies, all in flight while the
// warp polls q'.  Fast path (d' = 32, no threshold, no score outputs): per head, the staged rows are the M
// dimension of mma tiles, q' (split into bf16 hi + lo, ~16 bits) the columns; 16 spans x 1 head per 4 mma.
// General path: compact scalar loops from shared memory (the code footprint matters more than the
// arithmetic here: every item runs this once).
// ---------------------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ void route_item(const FusedParams& P, const Item& I, uint8_t* region, int lane,
                                           unsigned long long* tm) {
  const int bg = I.bg, g = bg % P.Hkv, dp = P.dp, lpr = dp >> 3;
  const int gid = lane >> 2, t4 = lane & 3;
  const int nsp = I.b - I.a;
  const uint8_t* route = (const uint8_t*)P.lv.route;
  const int total = nsp * G * lpr;
#pragma unroll 2
  for (int i = lane; i < total; i += 32) {
    const int c = i % lpr, t = i / lpr;
    const int hl = t / nsp, s = t - hl * nsp;
    cp_async16(region + (size_t)i * 16,
               route + ((size_t)(g * G + hl) * P.route_head_stride + (size_t)(I.span0 + I.a + s) * dp) * 2 + c * 16);
  }
  cp_async_commit();
  const float inv_sqrt_dp = rsqrtf((float)dp);
  uint32_t* gkeys = P.keys + (size_t)bg * P.keys_stride;
  const float* gqp = P.qp + (size_t)bg * G * dp;
  if (dp == 32 && P.tau == nullptr && P.logits_out == nullptr && P.alpha_out == nullptr) {
    uint32_t bh[4] = {0u, 0u, 0u, 0u}, bl[4] = {0u, 0u, 0u, 0u};
    float lnl[4];                                                // ln|S| of span 16 i + gid + 8 (t4 & 1)
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int s = 16 * i + gid + 8 * (t4 & 1);
      lnl[i] = s < nsp ? P.cv.ln_len[I.span0 + I.a + s] : 0.f;
    }
    if (gid < G) {
      const float4 v0 = poll_qp4(gqp + gid * 32 + 8 * t4), v1 = poll_qp4(gqp + gid * 32 + 8 * t4 + 4);
      split_bf16(v0.x * inv_sqrt_dp, v0.y * inv_sqrt_dp, bh[0], bl[0]);
      split_bf16(v0.z * inv_sqrt_dp, v0.w * inv_sqrt_dp, bh[1], bl[1]);
      split_bf16(v1.x * inv_sqrt_dp, v1.y * inv_sqrt_dp, bh[2], bl[2]);
      split_bf16(v1.z * inv_sqrt_dp, v1.w * inv_sqrt_dp, bh[3], bl[3]);
    }
    __syncwarp();
    mark(tm, 0, lane);
    cp_async_wait<0>();
    __syncwarp();
    mark(tm, 1, lane);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int s0 = 16 * i;
      if (s0 >= nsp) break;
      float Xa = -INFINITY, Xb = -INFINITY;                      // spans s0 + gid and s0 + gid + 8
#pragma unroll
      for (int hl = 0; hl < G; ++hl) {
        const uint8_t* ra = region + ((size_t)hl * nsp + s0 + gid) * 64 + t4 * 16;
        const uint4 a = *reinterpret_cast<const uint4*>(ra), c8 = *reinterpret_cast<const uint4*>(ra + 8 * 64);
        float c[4] = {0.f, 0.f, 0.f, 0.f};
        mma16816_full(c, a.x, c8.x, a.y, c8.y, bh[0], bh[1]);
        mma16816_full(c, a.z, c8.z, a.w, c8.w, bh[2], bh[3]);
        mma16816_full(c, a.x, c8.x, a.y, c8.y, bl[0], bl[1]);
        mma16816_full(c, a.z, c8.z, a.w, c8.w, bl[2], bl[3]);
        if (t4 == (hl >> 1)) {                                   // this lane holds column hl
          Xa = fmaxf(Xa, (hl & 1) ? c[1] : c[0]);
          Xb = fmaxf(Xb, (hl & 1) ? c[3] : c[2]);
        }
      }
      Xa = quad_max(Xa); Xb = quad_max(Xb);
      const int s = s0 + gid + 8 * (t4 & 1);
      if (t4 < 2 && s < nsp) gkeys[I.a + s] = order_key(((t4 & 1) ? Xb : Xa) + lnl[i]);
    }
    mark(tm, 2, lane);
    signal_ctr(grp_ctr(P, bg, C_ROUTE), lane);
    return;
  }
  float* sqp = reinterpret_cast<float*>(region + (size_t)P.route_spans * G * dp * 2);     // [G][dp]
  for (int i = 4 * lane; i < G * dp; i += 128) *reinterpret_cast<float4*>(sqp + i) = poll_qp4(gqp + i);
  mark(tm, 0, lane);
  cp_async_wait<0>();
  __syncwarp();
  mark(tm, 1, lane);
  for (int s = lane; s < nsp; s += 32) {
    const float lnl = P.cv.ln_len[I.span0 + I.a + s];
    float X = -INFINITY;
    bool elig = (P.tau == nullptr);
#pragma unroll 1
    for (int hl = 0; hl < G; ++hl) {
      const uint4* row = reinterpret_cast<const uint4*>(region + ((size_t)hl * nsp + s) * dp * 2);
      const float4* qv = reinterpret_cast<const float4*>(sqp + hl * dp);
      float acc = 0.f;
#pragma unroll 1
      for (int c = 0; c < lpr; ++c) {
        const uint4 v = row[c];
        const float4 q0 = qv[2 * c], q1 = qv[2 * c + 1];
        acc = fmaf(__uint_as_float(v.x << 16), q0.x, acc); acc = fmaf(__uint_as_float(v.x & 0xffff0000u), q0.y, acc);
        acc = fmaf(__uint_as_float(v.y << 16), q0.z, acc); acc = fmaf(__uint_as_float(v.y & 0xffff0000u), q0.w, acc);
        acc = fmaf(__uint_as_float(v.z << 16), q1.x, acc); acc = fmaf(__uint_as_float(v.z & 0xffff0000u), q1.y, acc);
        acc = fmaf(__uint_as_float(v.w << 16), q1.z, acc); acc = fmaf(__uint_as_float(v.w & 0xffff0000u), q1.w, acc);
      }
      const float x = fmaf(acc, inv_sqrt_dp, lnl);            // Eq. 5, pre-sigmoid logit
      const float a = 1.f / (1.f + __expf(-x));
      const int h = g * G + hl;
      if (P.logits_out) P.logits_out[(size_t)h * P.m_tot + I.span0 + I.a + s] = x;
      if (P.alpha_out) P.alpha_out[(size_t)h * P.m_tot + I.span0 + I.a + s] = a;
      if (P.tau != nullptr && a > P.tau[h]) elig = true;       // Eq. 9
      X = fmaxf(X, x);
    }
    gkeys[I.a + s] = elig ? order_key(X) : 0u;
  }
  mark(tm, 2, lane);
  signal_ctr(grp_ctr(P, bg, C_ROUTE), lane);
}

// ---------------------------------------------------------------------------------------------------
// a3 + a4 by a TEAM: the CTA's latency warps (the even warps, TS = 32 * ceil(nw / 2) threads) meet on named
// barrier 1 once the latency queue is exhausted and run selection and residency plan of the groups
// bg = blockIdx.x, + gridDim.x, ... together -- a single warp runs this serial chain at ~200 instructions
// per microsecond, and every expanded span of the group waits for it.  Tables live in the region of warp 0.
// ---------------------------------------------------------------------------------------------------
struct Team { int tt, ts, lane, tw, ntw; int* scratch; };

__device__ __forceinline__ void team_bar(const Team& T) { asm volatile("bar.sync 1, %0;" ::"r"(T.ts) : "memory"); }

// exclusive prefix sum over the team (two barriers); *total = sum over the team
__device__ __forceinline__ int team_excl_scan(const Team& T, int v, int* total) {
  const int ex = warp_excl_scan(v, T.lane);
  if (T.lane == 31) T.scratch[T.tw] = ex + v;
  team_bar(T);
  int base = 0, tot = 0;
  for (int w = 0; w < T.ntw; ++w) { const int c = T.scratch[w]; if (w < T.tw) base += c; tot += c; }
  team_bar(T);
  *total = tot;
  return base + ex;
}

// descending bitonic sort of n (power of two) 64-bit keys in shared memory by the team
__device__ __forceinline__ void bitonic_sort_desc_team(const Team& T, unsigned long long* keys, int n) {
  for (int size = 2; size <= n; size <<= 1) {
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int i = T.tt; i < (n >> 1); i += T.ts) {
        const int lo = ((i & ~(stride - 1)) << 1) | (i & (stride - 1));
        const int hi = lo | stride;
        const bool desc = ((lo & size) == 0);
        const unsigned long long a = keys[lo], c = keys[hi];
        if ((a < c) == desc) { keys[lo] = c; keys[hi] = a; }
      }
      team_bar(T);
    }
  }
}

// meta = |S| << 16 | rank_k | rank_v << 8 of the span
__device__ __forceinline__ void write_zdesc(const FusedParams& P, ZDescG* zd, int bg, int g, int span0, int id, uint32_t it,
                                            uint32_t meta, uint32_t epoch) {
  ZDescG d;
  d.src = 0ull; d.bytes = 0u; d.len_rr = 0u; d.way_miss = it; d.id = id; d.epoch0 = epoch; d.epoch1 = epoch;
  if (id >= 0) {
    const int gs = span0 + id;
    const int rr = (int)(meta & 0xffffu);
    const int len = (int)(meta >> 16);
    d.len_rr = meta;
    d.bytes = (uint32_t)blob_dims(2, len, rr & 0xff, (rr >> 8) & 0xff).bytes;
    const uint8_t* src = (it & 0x80000000u) ? P.host_arena + P.lv.dir_off[(size_t)g * P.spans_cap + gs]
                                            : P.lv.slots + ((size_t)bg * P.ways + (it & 0x3FFFFFFFu)) * P.slot_bytes;
    d.src = (unsigned long long)src;
  }
  uint4* o = reinterpret_cast<uint4*>(zd);
  o[0] = make_uint4((uint32_t)d.src, (uint32_t)(d.src >> 32), d.bytes, d.epoch0);
  o[1] = make_uint4(d.len_rr, d.way_miss, (uint32_t)d.id, d.epoch1);
}

struct PlanTables {
  int32_t* sh_ids; int16_t* way_of; int32_t* sh_tag; uint32_t* sh_stamp; int32_t* sh_victim; uint32_t* sh_mask;
  uint32_t* meta;      // [m] |S| << 16 | rank_k | rank_v << 8 of every span of the group
};
__device__ __forceinline__ PlanTables plan_tables(const FusedParams& P, uint8_t* region) {
  PlanTables t;
  t.sh_ids = reinterpret_cast<int32_t*>(region + P.sm_ids);
  t.way_of = reinterpret_cast<int16_t*>(region + P.sm_wayof);
  t.sh_tag = reinterpret_cast<int32_t*>(region + P.sm_tags);
  t.sh_stamp = reinterpret_cast<uint32_t*>(t.sh_tag + P.ways);
  t.sh_victim = reinterpret_cast<int32_t*>(t.sh_stamp + P.ways);
  t.sh_mask = reinterpret_cast<uint32_t*>(region + P.sm_mask);
  t.meta = reinterpret_cast<uint32_t*>(region + P.sm_meta);
  return t;
}

// first half of the plan: needs nothing from this step's routing, runs while the ROUTE items are in flight
__device__ __forceinline__ void plan_init_team(const FusedParams& P, const Team& T, const PlanTables& t, int bg, int span0,
                                               int m) {
  const int g = bg % P.Hkv;
  for (int s0 = 0; s0 < m; s0 += 8 * T.ts) {                   // 16 loads in flight per thread
    int len[8], rr[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int s = min(s0 + u * T.ts + T.tt, m - 1);
      len[u] = P.cv.span_len[span0 + s];
      rr[u] = P.lv.dir_rank[(size_t)g * P.spans_cap + span0 + s];
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int s = s0 + u * T.ts + T.tt;
      if (s < m) t.meta[s] = ((uint32_t)len[u] << 16) | (uint32_t)(rr[u] & 0xffff);
    }
  }
  const int32_t* tags = P.lv.tags + (size_t)bg * P.ways;
  const uint32_t* stamps = P.lv.stamps + (size_t)bg * P.ways;
  for (int w = T.tt; w < P.mask_words; w += T.ts) t.sh_mask[w] = 0u;
  for (int s = T.tt; s < m; s += T.ts) t.way_of[s] = (int16_t)-1;
  for (int w = T.tt; w < P.ways; w += T.ts) { t.sh_tag[w] = tags[w]; t.sh_stamp[w] = stamps[w]; t.sh_victim[w] = -1; }
  team_bar(T);
  for (int w = T.tt; w < P.ways; w += T.ts) { const int tg = t.sh_tag[w]; if (tg >= 0 && tg < m) t.way_of[tg] = (int16_t)w; }
  team_bar(T);
}

// a4: residency plan of (b, g).  The device factor cache of a (layer, sequence, kv head) is `ways` slots with
// a tag (span id) and a stamp (step of last use).  The first n_zoom entries of sh_ids are this step's zoom
// set: resident ones are hits, the others are demand misses and take the least-recently-used slots not
// needed by this step.  Entries n_zoom .. n_cand-1 are prefetch candidates (the next-best spans by routing
// score): the non-resident ones get a slot too and are copied by the side-stream prefetch kernel after
// this layer's kernel.  Also: zoom bit-mask for the coarse items (an expanded span's coarse entry is
// replaced by its tokens), de-duplication of caller-supplied ids, one descriptor per
// expanded span for the ZOOM items, statistics.
__device__ __forceinline__ void plan_team(const FusedParams& P, const Team& T, const PlanTables& t, int bg, int span0,
                                          int m, int n_zoom, int n_cand, bool dedupe, uint32_t epoch) {
  const int g = bg % P.Hkv, ways = P.ways;
  int32_t* tags = P.lv.tags + (size_t)bg * ways;
  uint32_t* stamps = P.lv.stamps + (size_t)bg * ways;
  uint32_t* items = P.lv.items + (size_t)bg * P.kc;
  int32_t* item_span = P.lv.item_span + (size_t)bg * P.kc;
  ZDescG* zd = P.zdesc + (size_t)bg * P.kc;
  const uint32_t cur = epoch;
  int n_hit = 0, n_miss = 0, n_pf = 0;
  unsigned long long bytes_algo = 0, bytes_h2d = 0;
  // pass 1: validate / de-duplicate, zoom mask, residency lookup
  for (int j = T.tt; j < n_cand; j += T.ts) {
    int id = t.sh_ids[j];
    if (id < 0 || id >= m) id = -1;
    const bool zoom = j < n_zoom;
    if (id >= 0 && zoom) {
      const uint32_t bit = 1u << (id & 31);
      const uint32_t old = atomicOr(&t.sh_mask[id >> 5], bit);
      if (dedupe && (old & bit)) id = -1;                      // duplicate of an id seen before: dropped
    }
    int way = -1;
    uint32_t meta = 0u;
    if (id >= 0) {
      way = t.way_of[id];
      if (way >= 0) t.sh_stamp[way] = cur;
      meta = t.meta[id];
      const int rk = meta & 0xff, rv = (meta >> 8) & 0xff;
      const int len = (int)(meta >> 16);
      const unsigned long long bb = blob_dims(2, len, rk, rv).bytes;
      if (zoom) {
        bytes_algo += (unsigned long long)(rk + rv) * (len + kD) * 2 + 4ull * (rk + rv);
        if (way >= 0) ++n_hit; else { ++n_miss; bytes_h2d += bb; }
      } else if (way < 0) { ++n_pf; bytes_h2d += bb; }
    }
    t.sh_ids[j] = id;
    item_span[j] = id;
    items[j] = (way >= 0) ? (uint32_t)way : 0xFFFFFFFFu;
    // hits (and dropped duplicates) publish their descriptor at once: the ZOOM items poll it and start
    // while the misses are still being given slots
    if (zoom && (way >= 0 || id < 0)) write_zdesc(P, zd + j, bg, g, span0, id, (uint32_t)max(way, 0), meta, epoch);
  }
  for (int j = n_zoom + T.tt; j < min(P.k_cap, m); j += T.ts) write_zdesc(P, zd + j, bg, g, span0, -1, 0u, 0u, epoch);
  int n_need;
  team_excl_scan(T, n_miss + n_pf, &n_need);                   // (its barriers also publish pass 1)
  n_need = min(n_need, ways);
  // victims: the n_need oldest ways not used by this step (ties to the lower way), by repeated extraction
  // of the minimum (stamp, way) -- only as many as this step has misses
  if (T.tw == 0) {
    for (int v = 0; v < n_need; ++v) {
      unsigned long long best = ~0ull;
      for (int w = T.lane; w < ways; w += 32)
        if (t.sh_stamp[w] != cur) best = min(best, ((unsigned long long)t.sh_stamp[w] << 32) | (unsigned long long)w);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) best = min(best, __shfl_xor_sync(0xffffffffu, best, o));
      if (best == ~0ull) break;
      const int w = (int)(best & 0xffffffffull);
      if (T.lane == 0) { t.sh_victim[v] = w; t.sh_stamp[w] = cur; }    // marked used: not extracted again
      __syncwarp();
    }
  }
  team_bar(T);
  // pass 2: misses take victims in item order; descriptors of the zoom set
  int miss_base = 0;
  for (int j0 = 0; j0 < n_cand; j0 += T.ts) {
    const int j = j0 + T.tt;
    const int id = (j < n_cand) ? t.sh_ids[j] : -1;
    uint32_t it = (j < n_cand) ? items[j] : 0u;
    const bool miss = id >= 0 && it == 0xFFFFFFFFu;
    int tot;
    const int off = team_excl_scan(T, miss ? 1 : 0, &tot);
    if (miss) {
      const int vi = miss_base + off;
      const int way = vi < ways ? t.sh_victim[vi] : -1;
      if (way >= 0) {
        t.sh_tag[way] = id;
        it = (uint32_t)way | 0x80000000u;
      } else {
        it = 0xC0000000u;                                      // no free slot: fetch, do not keep
      }
      items[j] = it;
    }
    miss_base += tot;
    if (miss && j < n_zoom) write_zdesc(P, zd + j, bg, g, span0, id, it, t.meta[id], epoch);
  }
  team_bar(T);
  for (int w = T.tt; w < ways; w += T.ts) { tags[w] = t.sh_tag[w]; stamps[w] = t.sh_stamp[w]; }
  uint32_t* gmask = P.lv.zoom_mask + (size_t)bg * P.mask_words;
  for (int w = T.tt; w < P.mask_words; w += T.ts) gmask[w] = t.sh_mask[w];
  if (T.tt == 0) { P.plan_counts[2 * bg] = n_zoom; P.plan_counts[2 * bg + 1] = n_cand; }
  team_bar(T);                                                 // every thread's global writes precede the release
  if (T.tt == 0) red_add_release(grp_ctr(P, bg, C_PLAN), 1);
  // statistics (off the critical path)
  n_hit = warp_sum_i(n_hit); n_miss = warp_sum_i(n_miss); n_pf = warp_sum_i(n_pf);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    bytes_algo += __shfl_xor_sync(0xffffffffu, bytes_algo, o);
    bytes_h2d += __shfl_xor_sync(0xffffffffu, bytes_h2d, o);
  }
  if (T.lane == 0) {
    if (n_hit) atomicAdd(&P.stats[ST_HITS], (unsigned long long)n_hit);
    if (n_miss) atomicAdd(&P.stats[ST_MISSES], (unsigned long long)n_miss);
    if (n_hit + n_miss) {
      atomicAdd(&P.stats[ST_ZOOMED], (unsigned long long)(n_hit + n_miss));
      atomicAdd(&P.stats[ST_SKIPPED], (unsigned long long)(n_hit + n_miss));
    }
    if (bytes_algo) atomicAdd(&P.stats[ST_FACTOR_ALGO], bytes_algo);
    if (bytes_h2d) atomicAdd(&P.stats[ST_H2D], bytes_h2d);
    if (n_pf) atomicAdd(&P.stats[ST_PREFETCHED], (unsigned long long)n_pf);
  }
}

// ---------------------------------------------------------------------------------------------------
// a3 (Eq. 9, cap L123): top-n_cand of the group's m keys.  A radix select (8 bits per pass, shared-memory
// histogram, starting at the highest bit in which the eligible keys differ) finds the n_cand-th largest
// key T; keys > T are taken, keys == T are taken in increasing span id until the count is met (ties to the
// lower id); the <= kc winners are then sorted by (key descending, id ascending).
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void select_team(const FusedParams& P, const Team& T, uint8_t* region, int bg, uint32_t epoch,
                                            unsigned long long* tm) {
  const int b = bg / P.Hkv;
  const int span0 = P.cv.seq_span_off[b];
  const int m = P.cv.seq_span_off[b + 1] - span0;
  const PlanTables t = plan_tables(P, region);
  if (P.mode & FM_ATTN) plan_init_team(P, T, t, bg, span0, m);
  if (!(P.mode & FM_ROUTE)) {
    // caller-supplied zoom set (sekv_decode_attn)
    int cnt = 0;
    if (P.ids != nullptr && P.count != nullptr) cnt = max(0, min(P.count[bg], P.k_cap));
    const int32_t* src = P.ids + (size_t)bg * max(P.k_cap, 1);
    for (int j = T.tt; j < cnt; j += T.ts) t.sh_ids[j] = src[j];
    team_bar(T);
    plan_team(P, T, t, bg, span0, m, cnt, cnt, true, epoch);
    return;
  }
  uint32_t* keys = reinterpret_cast<uint32_t*>(region);
  uint32_t* hist = reinterpret_cast<uint32_t*>(region + P.sm_hist);
  unsigned long long* cand = reinterpret_cast<unsigned long long*>(region + P.sm_cand);
  int* sel = T.scratch + 8;                // [0] digit, [1] keys above it, [2..4] ne / kmin / kmax, [5] keys == T, [6] slot
  for (int i = T.tt; i < 4 * 256; i += T.ts) hist[i] = 0u;     // one histogram per radix pass, zeroed while waiting
  const uint32_t* gkeys = P.keys + (size_t)bg * P.keys_stride;
  const int n_route = (m + P.route_spans - 1) / P.route_spans;
  if (T.tt == 0) {
    const int32_t* c = grp_ctr(P, bg, C_ROUTE);
    int v;
    for (;;) {
      asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(c) : "memory");
      if (v >= n_route) break;
      __nanosleep(64);
    }
    (void)ld_acquire(reinterpret_cast<const uint32_t*>(c));
    sel[2] = 0; sel[3] = -1; sel[4] = 0; sel[5] = 0; sel[6] = 0;
    mark(tm, 0, 0);
  }
  team_bar(T);
  for (int i = T.tt; i < (m + 3) / 4; i += T.ts) cp_async16(keys + 4 * i, gkeys + 4 * i);   // all in flight at once
  cp_async_commit();
  cp_async_wait<0>();
  team_bar(T);
  mark(tm, 1, T.tt);
  {
    int ne = 0;
    uint32_t kmin = 0xFFFFFFFFu, kmax = 0u;
    for (int i = T.tt; i < m; i += T.ts) {
      const uint32_t k = keys[i];
      if (k != 0u) { ++ne; kmin = min(kmin, k); kmax = max(kmax, k); }
    }
    ne = warp_sum_i(ne);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      kmin = min(kmin, __shfl_xor_sync(0xffffffffu, kmin, o));
      kmax = max(kmax, __shfl_xor_sync(0xffffffffu, kmax, o));
    }
    if (T.lane == 0) {
      atomicAdd(&sel[2], ne);
      atomicMin(reinterpret_cast<unsigned int*>(&sel[3]), kmin);
      atomicMax(reinterpret_cast<unsigned int*>(&sel[4]), kmax);
    }
  }
  team_bar(T);
  const int n_elig = sel[2];
  const uint32_t kmin = (uint32_t)sel[3], kmax = (uint32_t)sel[4];
  int cnt = P.k < 0 ? n_elig : min(P.k, n_elig);
  cnt = min(cnt, P.k_cap);
  int n_cand = cnt;
  if (P.k >= 0 && (P.mode & FM_ATTN)) n_cand = min(min(cnt + P.prefetch, n_elig), P.kc);
  uint32_t Tk = 0u;           // threshold key
  int need = 0;               // keys == Tk to take
  if (n_cand == 0) {
    Tk = 0xFFFFFFFFu;
  } else if (n_cand < n_elig) {
    // the eligible keys agree on every bit above the highest bit in which kmin and kmax differ: the passes
    // start there (float keys of one binade share 9 bits: a pass over them would pile every key -- and
    // every shared-memory atomic -- into one bin)
    const int hb = 31 - __clz((int)((kmin ^ kmax) | 1u));
    const int top = min(24, max(0, hb - 7));                    // first digit = bits [top, top + 8)
    uint32_t maskb = (top + 8 >= 32) ? 0u : ~((1u << (top + 8)) - 1u);
    uint32_t prefix = kmax & maskb;
    need = n_cand;
    uint32_t* hp = hist;
    for (int shift = top; shift >= 0; shift = (shift >= 8 ? shift - 8 : (shift > 0 ? 0 : -1)), hp += 256) {
      for (int i = T.tt; i < m; i += T.ts) {
        const uint32_t k = keys[i];
        if (k != 0u && (k & maskb) == prefix) atomicAdd(&hp[(k >> shift) & 255u], 1u);
      }
      team_bar(T);
      if (T.tw == 0) {
        int loc[8], tot = 0;
#pragma unroll
        for (int e = 0; e < 8; ++e) { loc[e] = (int)hp[255 - (8 * T.lane + e)]; tot += loc[e]; }
        int run = warp_excl_scan(tot, T.lane);     // matching keys in bins above this lane's bins
#pragma unroll
        for (int e = 0; e < 8; ++e) {
          if (run < need && run + loc[e] >= need) { sel[0] = 255 - (8 * T.lane + e); sel[1] = run; sel[5] = loc[e]; }
          run += loc[e];
        }
      }
      team_bar(T);
      need -= sel[1];
      prefix |= (uint32_t)sel[0] << shift;
      maskb |= 255u << shift;
    }
    Tk = prefix;
  }
  mark(tm, 2, T.tt);
  const bool cut_ties = (n_cand != 0 && n_cand < n_elig) && sel[5] != need;   // more keys == T than are taken
  if (!cut_ties) {
    // every key >= T is taken: append in any order (the sort below fixes the order)
    const uint32_t lo_key = (n_cand != 0 && n_cand < n_elig) ? Tk : (n_cand == 0 ? 0xFFFFFFFFu : 1u);
    if (n_cand != 0)
      for (int i = T.tt; i < m; i += T.ts) {
        const uint32_t k = keys[i];
        if (k >= lo_key) {
          const int pos = atomicAdd(&sel[6], 1);
          if (pos < P.kc) cand[pos] = ((unsigned long long)k << 32) | (unsigned long long)(0xFFFFFFFFu - (uint32_t)i);
        }
      }
    team_bar(T);
  } else {
  // ordered compaction: each thread owns a contiguous block of span ids
  const int per = (m + T.ts - 1) / T.ts;
  const int lo = min(m, T.tt * per), hi = min(m, lo + per);
  int gt = 0, eq = 0;
  for (int i = lo; i < hi; ++i) { const uint32_t k = keys[i]; gt += (k > Tk); eq += (k == Tk); }
  int dummy;
  const int eq_before = team_excl_scan(T, eq, &dummy);
  const int take_eq = (Tk == 0u) ? 0 : max(0, min(eq, need - eq_before));
  int pos = team_excl_scan(T, gt + take_eq, &dummy);
  int taken = 0;
  for (int i = lo; i < hi; ++i) {
    const uint32_t k = keys[i];
    bool s = k > Tk;
    if (k == Tk && taken < take_eq) { s = true; ++taken; }
    if (s && pos < P.kc) cand[pos++] = ((unsigned long long)k << 32) | (unsigned long long)(0xFFFFFFFFu - (uint32_t)i);
  }
  team_bar(T);
  }
  if (n_cand <= T.ts) {
    if (T.tt < n_cand) {
      const unsigned long long mine = cand[T.tt];
      int r = 0;
      for (int i = 0; i < n_cand; ++i) r += (cand[i] > mine);
      t.sh_ids[r] = (int32_t)(0xFFFFFFFFu - (uint32_t)(mine & 0xFFFFFFFFull));
    }
  } else {
    int n2 = 64;
    while (n2 < n_cand) n2 <<= 1;
    for (int j = n_cand + T.tt; j < n2; j += T.ts) cand[j] = 0ull;
    team_bar(T);
    bitonic_sort_desc_team(T, cand, n2);
    for (int j = T.tt; j < n_cand; j += T.ts) t.sh_ids[j] = (int32_t)(0xFFFFFFFFu - (uint32_t)(cand[j] & 0xFFFFFFFFull));
  }
  team_bar(T);
  mark(tm, 3, T.tt);
  int32_t* my_ids = P.ids + (size_t)bg * max(P.k_cap, 1);
  for (int j = T.tt; j < P.k_cap; j += T.ts) my_ids[j] = j < cnt ? t.sh_ids[j] : -1;
  if (T.tt == 0) P.count[bg] = cnt;
  if (P.mode & FM_ATTN) plan_team(P, T, t, bg, span0, m, cnt, n_cand, false, epoch);
}

// one partial record (m2, l, pad, pad, o[128]) per head; lane (gid, t4) holds head gid's (m, l) and the
// accumulators listed by the callers
__device__ __forceinline__ float* part_ptr(const FusedParams& P, const Item& I, int hl) {
  return P.partials + ((size_t)I.pbase + (size_t)hl * I.np + I.part) * kPartStride;
}

// ---------------------------------------------------------------------------------------------------
// a5: rows [I.a, I.b) of the entry table of (b, g): pool tokens (logit = q.K/sqrt(d)) and unexpanded coarse
// entries (logit = q.k_bar/sqrt(d) + ln|S|, value v_bar).  16-row tiles of K and V
// stream through a kStages-deep cp.async ring in the warp's region.  Shared-memory layout of a stage:
// K rows then V rows, 256 bytes per row, 16-byte chunk c of row r stored at chunk c ^ ((r & 1) << 2)
// (K) or c ^ (((r >> 1) & 3) << 1) (V): both fragment access patterns below are bank-conflict free.
//   QK^T : lane (gid = lane/4, t4 = lane%4) reads chunk (t4 + 4j) of the K row of token gid; its four
//          words are the (b0,b1) pairs of two k-steps; Q is loaded the same way (the contraction index
//          may be permuted consistently on both operands).
//   P V  : computed transposed, O^T = V^T P^T (M = 16 dims, N = 8 heads, K = 16 tokens): the C fragment
//          of S IS the B fragment of P^T.  P (fp32) is split into bf16 hi + lo parts and multiplied
//          twice, so probabilities carry ~16 bits.
// ---------------------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ void rows_item(const FusedParams& P, const Item& I, uint8_t* region, int lane, unsigned long long* tm) {
  const int bg = I.bg, b = bg / P.Hkv, g = bg % P.Hkv;
  const int gid = lane >> 2, t4 = lane & 3;
  const int A = I.A, row_begin = I.a, row_end = I.b;
  const uint8_t* Kb = (const uint8_t*)P.lv.ent_k + ((size_t)g * P.ent_head_stride + (size_t)I.row0 * kD) * 2;
  const uint8_t* Vb = (const uint8_t*)P.lv.ent_v + ((size_t)g * P.ent_head_stride + (size_t)I.row0 * kD) * 2;
  const float scale2 = rsqrtf((float)kD) * kLog2e;
  const int ntiles = (row_end - row_begin + 15) >> 4;

  // chunk idx = lane + 32 i of a 16 x 256-byte tile is row r = 2 i + (lane >> 4), 16-byte chunk c = lane & 15:
  // global offsets are contiguous and both swizzles are per-lane constants plus compile-time terms in i
  const int lr = lane >> 4, lc = lane & 15;
  const uint32_t dk0 = (uint32_t)(lr * 256 + ((lc ^ (lr << 2)) << 4));
  const uint32_t dv0 = (uint32_t)(lr * 256);
  auto fill = [&](int t) {
    uint8_t* Ks = region + (t % kStages) * kStageBytes;
    uint8_t* Vs = Ks + 16 * kD * 2;
    const int r0 = row_begin + t * 16;
    if (r0 + 16 <= row_end) {                                   // full tile: no clamping
      const size_t src = (size_t)r0 * (kD * 2) + lane * 16;
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        cp_async16(Ks + dk0 + 512 * i, Kb + src + 512 * i);
        cp_async16(Vs + dv0 + 512 * i + ((lc ^ ((i & 3) << 1)) << 4), Vb + src + 512 * i);
      }
    } else {
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int r = 2 * i + lr;
        const size_t src = (size_t)min(r0 + r, row_end - 1) * (kD * 2) + lc * 16;
        cp_async16(Ks + dk0 + 512 * i, Kb + src);
        cp_async16(Vs + dv0 + 512 * i + ((lc ^ ((i & 3) << 1)) << 4), Vb + src);
      }
    }
  };
#pragma unroll
  for (int t = 0; t < kStages; ++t) {
    if (t < ntiles) fill(t);
    cp_async_commit();
  }
  // biases of a COARSE item: lane L holds rows row_begin + L and row_begin + 32 + L.  EVERY coarse entry is
  // included (no dependency on this step's zoom set): the ZOOM item of an expanded span subtracts that span's
  // coarse term again (the softmax numerator and denominator are sums, "replaced by").
  float bias_reg[2] = {0.f, 0.f};
  if (I.kind == IT_COARSE) {
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int row = row_begin + 32 * u + lane;
      bias_reg[u] = row < row_end ? P.cv.ln_len[I.span0 + row - A] * kLog2e : -INFINITY;
    }
  }
  uint32_t qf[4][4];
  load_q_frags(P.q + ((size_t)b * P.Hq + (size_t)g * G) * kD, G, gid, t4, qf);
  float m_run = -INFINITY, l_run = 0.f;
  // acc[s][w][2o + c] = O[head 2*t4 + c][dim 64s + 8gid + 2w + o]
  float acc[2][4][4];
#pragma unroll
  for (int s = 0; s < 2; ++s)
#pragma unroll
    for (int w = 0; w < 4; ++w) { acc[s][w][0] = 0.f; acc[s][w][1] = 0.f; acc[s][w][2] = 0.f; acc[s][w][3] = 0.f; }

  for (int t = 0; t < ntiles; ++t) {
    cp_async_wait<kStages - 1>();
    __syncwarp();
    const uint8_t* Ks = region + (t % kStages) * kStageBytes;
    const uint8_t* Vs = Ks + 16 * kD * 2;
    const int r0 = row_begin + t * 16;
    float sacc[2][4];
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) {
      sacc[nt][0] = sacc[nt][1] = sacc[nt][2] = sacc[nt][3] = 0.f;
      const int r = 8 * nt + gid;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const uint4 kv = *reinterpret_cast<const uint4*>(Ks + r * 256 + (((t4 + 4 * j) ^ ((r & 1) << 2)) << 4));
        mma16816(sacc[nt], qf[j][0], qf[j][1], kv.x, kv.y);
        mma16816(sacc[nt], qf[j][2], qf[j][3], kv.z, kv.w);
      }
    }
    // logits in the base-2 domain with the entry bias (0 for pool tokens, ln|S| for coarse entries,
    // -inf for expanded spans and for rows past the item)
    float z[2][2];
    if (I.kind == IT_POOL && r0 + 16 <= row_end) {     // warp-uniform fast path
#pragma unroll
      for (int nt = 0; nt < 2; ++nt) { z[nt][0] = sacc[nt][0] * scale2; z[nt][1] = sacc[nt][1] * scale2; }
    } else {
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int ri = 16 * t + 8 * nt + 2 * t4 + e;      // row index within the item
          float bias = 0.f;
          if (I.kind == IT_COARSE) {
            const float b0 = __shfl_sync(0xffffffffu, bias_reg[0], ri & 31);
            const float b1 = __shfl_sync(0xffffffffu, bias_reg[1], ri & 31);
            bias = (ri < 32) ? b0 : b1;
          }
          if (row_begin + ri >= row_end) bias = -INFINITY;
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
      uint4 vf[4];
#pragma unroll
      for (int rr = 0; rr < 4; ++rr) {
        const int r = 2 * t4 + (rr & 1) + 8 * (rr >> 1);
        vf[rr] = *reinterpret_cast<const uint4*>(Vs + r * 256 + (((gid + 8 * s) ^ (t4 << 1)) << 4));
      }
      const uint32_t ra[4] = {vf[0].x, vf[0].y, vf[0].z, vf[0].w};
      const uint32_t rb[4] = {vf[1].x, vf[1].y, vf[1].z, vf[1].w};
      const uint32_t rc[4] = {vf[2].x, vf[2].y, vf[2].z, vf[2].w};
      const uint32_t rd[4] = {vf[3].x, vf[3].y, vf[3].z, vf[3].w};
#pragma unroll
      for (int w = 0; w < 4; ++w) {
        const uint32_t a0 = __byte_perm(ra[w], rb[w], 0x5410), a1 = __byte_perm(ra[w], rb[w], 0x7632);
        const uint32_t a2 = __byte_perm(rc[w], rd[w], 0x5410), a3 = __byte_perm(rc[w], rd[w], 0x7632);
        mma16816_full(acc[s][w], a0, a1, a2, a3, b0h, b1h);
        mma16816_full(acc[s][w], a0, a1, a2, a3, b0l, b1l);
      }
    }
    __syncwarp();                                      // every lane is done with this stage
    if (t + kStages < ntiles) fill(t + kStages);
    cp_async_commit();
  }
  cp_async_wait<0>();
  l_run = quad_sum(l_run);
  if (gid < G && t4 == 0) {
    float* pp = part_ptr(P, I, gid);
    pp[0] = m_run; pp[1] = l_run;
  }
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    const int hh = 2 * t4 + c;
    if (hh < G) {
      float* o = part_ptr(P, I, hh) + 4;
#pragma unroll
      for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int w = 0; w < 4; ++w)
          *reinterpret_cast<float2*>(o + 64 * s + 8 * gid + 2 * w) = make_float2(acc[s][w][c], acc[s][w][2 + c]);
    }
  }
  __syncwarp();
  if (lane == 0) {
    red_add_release(grp_ctr(P, bg, C_EARLY), 1);
    red_add_release(grp_ctr(P, bg, C_ATTN), 1);
  }
}

// ---------------------------------------------------------------------------------------------------
// a6: one expanded span, blob resident in the warp's region; the warp walks its 16-token chunks.
//   c = sigma_K o (Vt_K q) * log2e/sqrt(d)   (rows of Vt_K play the role of tokens in QK^T)
//   logits = U_K c  (= (U Sigma V^T q), Eq. 8 never materialised), p = 2^(z - m)
//   y = p^T U_V,   o += (sigma_V o y) V_V^T  accumulated into the warp's running (M, L, of)
// ---------------------------------------------------------------------------------------------------
// NK: compile-time bound on the 16-wide k-steps over the key and value ranks (1, 2 or 4)
template <int G, int NK>
__device__ __forceinline__ void zoom_span_warp(const uint8_t* blob, const BlobDims& bd, int lane,
                                               const uint32_t (&qf)[4][4], float& M, float& L, float (&of)[16][4]) {
  const int gid = lane >> 2, t4 = lane & 3;
  const float* sK = (const float*)(blob + bd.off_sk);
  const float* sV = (const float*)(blob + bd.off_sv);
  const uint8_t* VtK = blob + bd.off_vtk;
  const uint8_t* VV = blob + bd.off_vv;
  const int nks = (bd.rkp + 15) >> 4, nvs = (bd.rvp + 15) >> 4;     // k-steps over the key / value rank
  const int ngrp = bd.lenp >> 4;
  const float scale2 = rsqrtf((float)kD) * kLog2e;
  // 1. c
  uint32_t ckh[NK][2], ckl[NK][2];
#pragma unroll
  for (int ks = 0; ks < NK; ++ks) {
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
  float yf[2 * NK][4];
#pragma unroll
  for (int n = 0; n < 2 * NK; ++n) { yf[n][0] = yf[n][1] = yf[n][2] = yf[n][3] = 0.f; }
  // two 16-token chunks per iteration: their logits are independent, one running-max update serves both
  for (int grp = 0; grp < ngrp; grp += 2) {
    const bool two = grp + 1 < ngrp;
    float sacc[2][2][4];
#pragma unroll
    for (int cc = 0; cc < 2; ++cc) {
      const uint8_t* UKc = blob + bd.off_chunks + (size_t)(grp + cc) * bd.chunk_bytes;
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        sacc[cc][u][0] = sacc[cc][u][1] = sacc[cc][u][2] = sacc[cc][u][3] = 0.f;
        const uint8_t* prow = UKc + (size_t)pi_index(u, gid) * (bd.rkp * 2) + t4 * 8;
#pragma unroll
        for (int ks = 0; ks < NK; ++ks) {
          if (ks < nks) {
            uint2 bv = make_uint2(0u, 0u);
            if ((cc == 0 || two) && 16 * ks + 4 * t4 < bd.rkp) bv = *reinterpret_cast<const uint2*>(prow + ks * 32);
            mma16816(sacc[cc][u], ckh[ks][0], ckh[ks][1], bv.x, bv.y);
            mma16816(sacc[cc][u], ckl[ks][0], ckl[ks][1], bv.x, bv.y);
          }
        }
      }
    }
    // this lane: head gid, tokens 16 (grp + cc) + 4*t4 + 2u + e
    float z[2][2][2];
    float mx = -INFINITY;
#pragma unroll
    for (int cc = 0; cc < 2; ++cc)
#pragma unroll
      for (int u = 0; u < 2; ++u)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          z[cc][u][e] = (16 * (grp + cc) + 4 * t4 + 2 * u + e < bd.len) ? sacc[cc][u][e] : -INFINITY;
          mx = fmaxf(mx, z[cc][u][e]);
        }
    mx = quad_max(mx);
    const float m_new = fmaxf(m_s, mx);
    const float m_safe = (m_new == -INFINITY) ? 0.f : m_new;
    if (__any_sync(0xffffffffu, m_new > m_s)) {
      const float corr = exp2f(m_s - m_safe);
      l_s *= corr;
#pragma unroll
      for (int n = 0; n < 2 * NK; ++n) { yf[n][0] *= corr; yf[n][1] *= corr; }
    }
    m_s = m_new;
#pragma unroll
    for (int cc = 0; cc < 2; ++cc) {
      if (cc == 1 && !two) break;
      const uint8_t* UVtc = blob + bd.off_chunks + (size_t)(grp + cc) * bd.chunk_bytes + bd.uvt_in_chunk;
      const float p00 = exp2f(z[cc][0][0] - m_safe), p01 = exp2f(z[cc][0][1] - m_safe);
      const float p10 = exp2f(z[cc][1][0] - m_safe), p11 = exp2f(z[cc][1][1] - m_safe);
      l_s += (p00 + p01) + (p10 + p11);
      uint32_t a0h, a0l, a2h, a2l;
      split_bf16(p00, p01, a0h, a0l);     // tokens 4*t4 + {0,1}  <-> k = 2*t4 + e
      split_bf16(p10, p11, a2h, a2l);     // tokens 4*t4 + {2,3}  <-> k = 8 + 2*t4 + e
      // y += P U_V : B[k = token][n = i] read from the transposed factor UVt[i][token]
#pragma unroll
      for (int n = 0; n < 2 * NK; ++n) {
        if (n < 2 * nvs) {
          const int irow = pi_index(n, gid);
          uint2 bv = make_uint2(0u, 0u);
          if (irow < bd.rvp) bv = *reinterpret_cast<const uint2*>(UVtc + (size_t)irow * (kLenPad * 2) + t4 * 8);
          mma16816(yf[n], a0h, a2h, bv.x, bv.y);
          mma16816(yf[n], a0l, a2l, bv.x, bv.y);
        }
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
  uint32_t yh[NK][2], yl[NK][2];          // yf[n][e] is head gid, rank index 16(n>>1) + 4*t4 + 2(n&1) + e
#pragma unroll
  for (int ks = 0; ks < NK; ++ks) {
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
    for (int ks = 0; ks < NK; ++ks) {
      if (ks < nvs) {
        uint2 bv = make_uint2(0u, 0u);
        if (16 * ks + 4 * t4 < bd.rvp) bv = *reinterpret_cast<const uint2*>(prow + ks * 32);
        mma16816(of[nd], yh[ks][0], yh[ks][1], bv.x, bv.y);
        mma16816(of[nd], yl[ks][0], yl[ks][1], bv.x, bv.y);
      }
    }
  }
}

__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }

// lane 0 starts a 1-D bulk copy into the warp's region; every lane waits for its bytes
__device__ __forceinline__ void region_fetch(uint8_t* region, const void* src, uint32_t bytes, uint64_t* bar,
                                             uint32_t& phase, int lane) {
  __syncwarp();                                    // every lane is done with the region's previous contents
  if (lane == 0) {
    fence_proxy_async_all();
    mbar_arrive_expect_tx(bar, bytes);
    bulk_g2s(region, src, bytes, bar);
  }
  mbar_wait(bar, phase);
  phase ^= 1u;
}

// poll a descriptor until both halves carry this launch's stamp
__device__ __forceinline__ ZDescG poll_zdesc(const ZDescG* p, uint32_t epoch) {
  uint4 a, c;
  for (;;) {
    asm volatile("ld.relaxed.gpu.global.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w) : "l"(p) : "memory");
    asm volatile("ld.relaxed.gpu.global.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(c.x), "=r"(c.y), "=r"(c.z), "=r"(c.w) : "l"(reinterpret_cast<const uint4*>(p) + 1) : "memory");
    if (a.w == epoch && c.w == epoch) break;
    __nanosleep(64);
  }
  ZDescG d;
  d.src = (unsigned long long)a.x | ((unsigned long long)a.y << 32);
  d.bytes = a.z; d.epoch0 = a.w; d.len_rr = c.x; d.way_miss = c.y; d.id = (int32_t)c.z; d.epoch1 = c.w;
  return d;
}

// ---------------------------------------------------------------------------------------------------
// a4 + a6: plan items [I.a, I.b) of (b, g), one expanded span after the other through the warp's region
// ---------------------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ void zoom_item(const FusedParams& P, const Item& I, uint8_t* region, uint64_t* bar,
                                          uint32_t& phase, int lane, uint32_t epoch, unsigned long long* tm) {
  const int bg = I.bg, b = bg / P.Hkv, g = bg % P.Hkv;
  const int gid = lane >> 2, t4 = lane & 3;
  uint32_t qf[4][4];
  load_q_frags(P.q + ((size_t)b * P.Hq + (size_t)g * G) * kD, G, gid, t4, qf);
  const int j0 = I.a, j1 = I.b;                       // the plan stamps every descriptor of the schedule (id -1 = none)
  float M = -INFINITY, L = 0.f;
  float of[16][4];
#pragma unroll
  for (int n = 0; n < 16; ++n) { of[n][0] = of[n][1] = of[n][2] = of[n][3] = 0.f; }
  const ZDescG* zd = P.zdesc + (size_t)bg * P.kc;
  for (int j = j0; j < j1; ++j) {
    const ZDescG d = poll_zdesc(zd + j, epoch);
    if (j == j0) mark(tm, 0, lane);
    if (d.id < 0) continue;
    // the span's coarse entry (k_bar, v_bar, ln|S|) was counted by a COARSE item: loads for taking it out again
    const size_t crow = ((size_t)g * P.ent_head_stride + (size_t)(I.row0 + I.A + d.id) * kD) * 2;
    const uint8_t* kbar = (const uint8_t*)P.lv.ent_k + crow;
    const uint8_t* vbar = (const uint8_t*)P.lv.ent_v + crow;
    uint4 kc4[4];
    uint32_t vb[16];
#pragma unroll
    for (int jj = 0; jj < 4; ++jj) kc4[jj] = gid == 0 ? ldg16(kbar + (t4 + 4 * jj) * 16) : make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
    for (int nd = 0; nd < 16; ++nd) vb[nd] = __ldg(reinterpret_cast<const uint32_t*>(vbar + (8 * nd + 2 * t4) * 2));
    const float lnl2 = P.cv.ln_len[I.span0 + d.id] * kLog2e;
    region_fetch(region, (const void*)d.src, d.bytes, bar, phase, lane);
    if (j == j0) mark(tm, 1, lane);
    const BlobDims bd = blob_dims(2, (int)(d.len_rr >> 16), d.len_rr & 0xff, (d.len_rr >> 8) & 0xff);
    const int kst = (max(bd.rkp, bd.rvp) + 15) >> 4;
    if (kst <= 1) zoom_span_warp<G, 1>(region, bd, lane, qf, M, L, of);
    else if (kst == 2) zoom_span_warp<G, 2>(region, bd, lane, qf, M, L, of);
    else zoom_span_warp<G, 4>(region, bd, lane, qf, M, L, of);
    {
      // minus the coarse entry: logit z = q.k_bar/sqrt(d) + ln|S| exactly as the COARSE item computed it
      float sacc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int jj = 0; jj < 4; ++jj) {
        mma16816(sacc, qf[jj][0], qf[jj][1], kc4[jj].x, kc4[jj].y);
        mma16816(sacc, qf[jj][2], qf[jj][3], kc4[jj].z, kc4[jj].w);
      }
      const float zc = __shfl_sync(0xffffffffu, sacc[0], lane & ~3);     // column 0 (the entry) of head gid
      const float z = fmaf(zc, rsqrtf((float)kD) * kLog2e, lnl2);
      const float M_new = fmaxf(M, z);
      const float c_old = exp2f(M - M_new), w = exp2f(z - M_new);
      M = M_new;
      L = L * c_old - (t4 == 0 ? w : 0.f);                               // L is summed over the quad at the end
#pragma unroll
      for (int nd = 0; nd < 16; ++nd) {
        of[nd][0] = fmaf(-w, __uint_as_float(vb[nd] << 16), of[nd][0] * c_old);
        of[nd][1] = fmaf(-w, __uint_as_float(vb[nd] & 0xffff0000u), of[nd][1] * c_old);
      }
    }
    if (j == j0) mark(tm, 2, lane);
    if ((d.way_miss & 0xC0000000u) == 0x80000000u) {   // demand miss: the blob came over PCIe; keep it in its slot
      int4* dst = reinterpret_cast<int4*>(P.lv.slots + ((size_t)bg * P.ways + (d.way_miss & 0x3FFFFFFFu)) * P.slot_bytes);
      const int4* src = reinterpret_cast<const int4*>(region);
      for (int i = lane; i < (int)(d.bytes >> 4); i += 32) dst[i] = src[i];
    }
  }
  mark(tm, 3, lane);
  L = quad_sum(L);
  if (gid < G) {                                       // of[nd][c] is head gid, dimension 8*nd + 2*t4 + c
    float* pp = part_ptr(P, I, gid);
    if (t4 == 0) { pp[0] = M; pp[1] = L; }
#pragma unroll
    for (int nd = 0; nd < 16; ++nd) *reinterpret_cast<float2*>(pp + 4 + 8 * nd + 2 * t4) = make_float2(of[nd][0], of[nd][1]);
  }
  signal_ctr(grp_ctr(P, bg, C_ATTN), lane);
}

// ---------------------------------------------------------------------------------------------------
// a7 (L61): log-sum-exp merge of the np partials of one query head -> out, lse.  The head's records are
// contiguous; they move into the warp's region by bulk copies and are reduced from shared memory.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void combine_item(const FusedParams& P, const Item& I, uint8_t* region, uint64_t* bar,
                                             uint32_t& phase, int lane, unsigned long long* tm) {
  const int bg = I.bg, b = bg / P.Hkv, g = bg % P.Hkv, hl = I.a, np = I.np;
  const int G = P.Hq / P.Hkv;
  const float* src = P.partials + ((size_t)I.pbase + (size_t)hl * np) * kPartStride;
  const int cap = P.region_bytes / (kPartStride * 4);
  const float* rec = reinterpret_cast<const float*>(region);
  float M = -INFINITY, L = 0.f;
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  // two phases: the POOL and COARSE partials (slots [0, I.b)) are complete long before the expanded spans
  // are; they are merged while those are still running, so only the ZOOM partials remain for the tail
  const int n_pool = I.b;
  wait_ctr(grp_ctr(P, bg, C_EARLY), n_pool, lane, nullptr);
  bool second = false;
  for (int p0 = 0; p0 < np; p0 += cap) {
    if (!second && p0 >= n_pool) { wait_ctr(grp_ctr(P, bg, C_ATTN), np, lane, tm); second = true; }
    const int n = min(cap, (second ? np : n_pool) - p0);
    region_fetch(region, src + (size_t)p0 * kPartStride, (uint32_t)(n * kPartStride * 4), bar, phase, lane);
    float mc = -INFINITY;
    for (int p = lane; p < n; p += 32) mc = fmaxf(mc, rec[p * kPartStride]);
    mc = warp_max(mc);
    const float Mn = fmaxf(M, mc);
    const float safe = (Mn == -INFINITY) ? 0.f : Mn;
    const float c_old = exp2f(M - safe);
    // weights in parallel (lane p), kept in the record's pad word; L by a warp reduction
    float lsum = 0.f;
    for (int p = lane; p < n; p += 32) {
      const float mp = rec[p * kPartStride];
      const float w = (mp == -INFINITY) ? 0.f : exp2f(mp - safe);
      const_cast<float*>(rec)[p * kPartStride + 2] = w;
      lsum = fmaf(rec[p * kPartStride + 1], w, lsum);
    }
    L = fmaf(L, c_old, warp_sum(lsum));
    acc.x *= c_old; acc.y *= c_old; acc.z *= c_old; acc.w *= c_old;
    __syncwarp();
#pragma unroll 4
    for (int p = 0; p < n; ++p) {
      const float w = rec[p * kPartStride + 2];
      const float4 v = reinterpret_cast<const float4*>(rec + p * kPartStride + 4)[lane];
      acc.x = fmaf(v.x, w, acc.x); acc.y = fmaf(v.y, w, acc.y); acc.z = fmaf(v.z, w, acc.z); acc.w = fmaf(v.w, w, acc.w);
    }
    M = Mn;
    if (!second && p0 + n >= n_pool) { p0 = n_pool - cap; }     // next round starts at the first non-POOL partial
  }
  if (!second) wait_ctr(grp_ctr(P, bg, C_ATTN), np, lane, tm);  // (no ZOOM / COARSE partials at all)
  const float inv = L > 0.f ? 1.f / L : 0.f;
  const size_t oi = ((size_t)b * P.Hq + (size_t)g * G + hl) * kD + 4 * lane;
  if (P.out_bf16) {
    uint2 o;
    o.x = pack_bf16(acc.x * inv, acc.y * inv);
    o.y = pack_bf16(acc.z * inv, acc.w * inv);
    *reinterpret_cast<uint2*>(reinterpret_cast<__nv_bfloat16*>(P.out) + oi) = o;
  } else {
    *reinterpret_cast<float4*>(reinterpret_cast<float*>(P.out) + oi) = make_float4(acc.x * inv, acc.y * inv, acc.z * inv, acc.w * inv);
  }
  if (P.lse && lane == 0) P.lse[b * P.Hq + g * G + hl] = L > 0.f ? (M + log2f(L)) * kLn2 : -INFINITY;
}

__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}

__device__ __forceinline__ Item load_item(const Item* p) {
  const uint4* s = reinterpret_cast<const uint4*>(p);
  const uint4 a = __ldg(s), c = __ldg(s + 1), d = __ldg(s + 2);
  Item I;
  I.kind = (int32_t)a.x; I.bg = (int32_t)a.y; I.a = (int32_t)a.z; I.b = (int32_t)a.w;
  I.part = (int32_t)c.x; I.A = (int32_t)c.y; I.row0 = (int32_t)c.z; I.span0 = (int32_t)c.w;
  I.pbase = (int32_t)d.x; I.np = (int32_t)d.y; I.pad0 = 0; I.pad1 = 0;
  return I;
}

template <int G>
__global__ void __maxnreg__(240) fused_layer_kernel(const __grid_constant__ FusedParams P) {
  extern __shared__ __align__(128) uint8_t dsm[];
  __shared__ uint64_t bars[8];
  __shared__ int last_flag;
  __shared__ unsigned long long tmid_s[8 * 4];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nw = blockDim.x >> 5;
  // Programmatic dependent launch: the next layer's grid may be scheduled as soon as this one's CTAs leave
  // their SMs (its CTAs then sit in the wait below), which hides the launch latency between the dependent
  // kernels of a step; everything this kernel touches is ordered after the previous grid by the wait.
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
  uint8_t* region = dsm + (size_t)warp * P.region_bytes;
  uint64_t* bar = &bars[warp];
  const uint32_t epoch = *reinterpret_cast<volatile const uint32_t*>(P.lv.layer_step) + 1u;
  if (lane == 0) {
    mbar_init(bar, 1);
    mbar_fence_init();
  }
  __syncwarp();
  uint32_t phase = 0u;
  unsigned long long* tm = P.trace ? &tmid_s[warp * 4] : nullptr;

  // Latency items are handed out statically to the first warps of the grid (every warp of a CTA takes one), so
  // the whole latency queue starts at t = 0; what is left of it (large batches) is claimed by the even warps,
  // which also form the CTA's selection / plan team.  Everything else is claimed from the main queue.
  const int nlw = (nw + 1) >> 1;
  const int total_w = (int)gridDim.x * nw, gw = (int)blockIdx.x * nw + warp;
  const bool team_member = (warp & 1) == 0;
  bool in_lat = false;
  __shared__ int team_scratch[16];
  // selection and residency plan of this CTA's groups by the team of latency warps (once per warp)
  auto team_work = [&]() {
    Team T;
    T.tt = (warp >> 1) * 32 + lane; T.ts = nlw * 32; T.lane = lane; T.tw = warp >> 1; T.ntw = nlw; T.scratch = team_scratch;
    team_bar(T);                                               // warp 0 is done with its region (the tables live there)
    for (int bg = (int)blockIdx.x; bg < P.BG; bg += (int)gridDim.x) {
      unsigned long long t0 = 0ull;
      if (P.trace) { t0 = globaltimer_ns(); if (T.tt == 0) { tm[0] = t0; tm[1] = t0; tm[2] = t0; tm[3] = t0; } }
      select_team(P, T, dsm, bg, epoch, tm);
      const int rec = P.main_end + bg;                         // trace record after the queue items
      if (P.trace && T.tt == 0 && rec < P.trace_cap) {
        unsigned long long* r = P.trace + 8 * (size_t)rec;
        r[0] = (unsigned long long)(uint32_t)IT_SELECT | ((unsigned long long)(uint32_t)bg << 32);
        r[1] = (unsigned long long)blockIdx.x;
        r[2] = t0; r[3] = globaltimer_ns();
        r[4] = tm[0]; r[5] = tm[1]; r[6] = tm[2]; r[7] = tm[3];
      }
      team_bar(T);
    }
  };
  auto claim = [&]() -> int {
    int i = 0;
    if (in_lat) {
      if (lane == 0) i = P.lat_begin + total_w + atomicAdd(P.ctrs, 1);
      i = __shfl_sync(0xffffffffu, i, 0);
      if (i < P.lat_end) return i;
      in_lat = false;
      team_work();
    }
    if (lane == 0) i = P.lat_end + atomicAdd(P.ctrs + 1, 1);
    return __shfl_sync(0xffffffffu, i, 0);
  };
  int idx;
  if (gw < P.lat_end - P.lat_begin) {
    idx = P.lat_begin + gw;
    in_lat = team_member;
  } else {
    if (team_member) team_work();
    idx = claim();
  }
  if (idx < P.main_end) {
    // Claims run ahead only through POOL items (no dependencies, nobody waits on one in particular): the
    // item after a POOL item is claimed, and its descriptor loaded, while the POOL item is processed.  Any
    // other item is claimed when the warp is free to run it, so it never waits behind a slow item.
    auto claim_after = [&](int just) -> int { return (!in_lat && just < P.pool_end) ? claim() : -1; };
    Item cur = load_item(P.items + idx);
    int nidx = claim_after(idx);
    for (;;) {
      const bool has_next = nidx >= 0 && nidx < P.main_end;
      Item nxt = cur;
      int nnidx = nidx;
      if (has_next) {
        nxt = load_item(P.items + nidx);
        nnidx = claim_after(nidx);
      }
      unsigned long long t0 = 0ull;
      const int cur_idx = idx;
      if (P.trace) { t0 = globaltimer_ns(); if (lane == 0) { tm[0] = t0; tm[1] = t0; tm[2] = t0; tm[3] = t0; } }
      switch (cur.kind) {
        case IT_QPROJ: qproj_item<G>(P, cur, lane); break;
        case IT_ROUTE: route_item<G>(P, cur, region, lane, tm); break;
        case IT_POOL:
        case IT_COARSE: rows_item<G>(P, cur, region, lane, tm); break;
        case IT_ZOOM: zoom_item<G>(P, cur, region, bar, phase, lane, epoch, tm); break;
        default: combine_item(P, cur, region, bar, phase, lane, tm); break;
      }
      if (P.trace && lane == 0 && cur_idx < P.trace_cap) {
        unsigned int smid;
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        unsigned long long* r = P.trace + 8 * (size_t)cur_idx;
        r[0] = (unsigned long long)(uint32_t)cur.kind | ((unsigned long long)(uint32_t)cur.bg << 32);
        r[1] = (unsigned long long)(smid & 0xffffu) | ((unsigned long long)(uint32_t)warp << 16);
        r[2] = t0; r[3] = globaltimer_ns();
        r[4] = tm[0]; r[5] = tm[1]; r[6] = tm[2]; r[7] = tm[3];
      }
      if (nidx < 0) {
        nidx = claim();
        if (nidx >= P.main_end) break;
        cur = load_item(P.items + nidx);
        idx = nidx;
        nidx = claim_after(idx);
        continue;
      }
      if (!has_next) break;
      cur = nxt;
      idx = nidx;
      nidx = nnidx;
    }
  }
  // an exiting warp has nothing left to claim, and the tail of the kernel is latency-bound: pull the tables
  // that head the next layer's dependency chain (W, routing summaries) into L2 while HBM is idle
  if (P.next_W != nullptr) {
    const size_t w_lines = P.next_W_bytes >> 7, r_lines = P.next_route_head_bytes >> 7;
    for (size_t i = (size_t)gw * 32 + lane; i < w_lines; i += (size_t)total_w * 32)
      asm volatile("prefetch.global.L2 [%0];" ::"l"(P.next_W + (i << 7)));
    for (size_t i = (size_t)gw * 32 + lane; i < r_lines * P.Hq; i += (size_t)total_w * 32) {
      const size_t h = i / r_lines, li = i - h * r_lines;
      asm volatile("prefetch.global.L2 [%0];" ::"l"(P.next_route + h * P.route_head_stride * 2 + (li << 7)));
    }
  }
  // last CTA out re-arms the queues and counters and advances the layer's step stamp
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    const int old = atomicAdd(P.ctrs + 2, 1);
    last_flag = (old == (int)gridDim.x - 1);
  }
  __syncthreads();
  if (last_flag) {
    __threadfence();
    for (int i = tid; i < 4 + 4 * P.BG; i += blockDim.x) P.ctrs[i] = 0;
    if (P.mode & FM_ROUTE)
      for (int i = tid; i < P.BG * G * P.dp; i += blockDim.x) reinterpret_cast<uint32_t*>(P.qp)[i] = kQpSentinel;
    if (tid == 0 && (P.mode & FM_ATTN)) {
      *P.lv.layer_step = epoch;
      atomicAdd(&P.stats[ST_LAYER_STEPS], 1ull);
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
  if (id < 0 || (it & 0xC0000000u) != 0x80000000u) return;
  if (threadIdx.x == 0) {
    const int way = (int)(it & 0x3FFFFFFFu);
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
static int pow2_ceil(int x) { int p = 1; while (p < x) p <<= 1; return p; }

// byte offsets of the select / plan tables inside a warp's region; returns the bytes they need
size_t fused_plan_smem(const sekv_handle* h, FusedParams* P) {
  const sekv_config& c = h->cfg;
  const int kc = std::max(c.k_cap, 1) + std::max(c.prefetch, 0);
  size_t o = (size_t)round_up(std::max(h->max_m, 1), 4) * 4;             // keys
  o = round_up_sz(o, 16); P->sm_hist = (int)o; o += 4 * 256 * 4;
  o = round_up_sz(o, 16); P->sm_cand = (int)o; o += (size_t)pow2_ceil(std::max(kc, 64)) * 8;
  o = round_up_sz(o, 16); P->sm_ids = (int)o; o += (size_t)kc * 4;
  o = round_up_sz(o, 16); P->sm_wayof = (int)o; o += (size_t)round_up(std::max(h->max_m, 1), 8) * 2;
  o = round_up_sz(o, 16); P->sm_tags = (int)o; o += (size_t)c.cache_ways * 12;
  o = round_up_sz(o, 16); P->sm_mask = (int)o; o += (size_t)h->mask_words * 4;
  o = round_up_sz(o, 16); P->sm_meta = (int)o; o += (size_t)round_up(std::max(h->max_m, 1), 4) * 4;
  return o;
}

// per-warp region: the rows ring, one factor blob, or the select / plan tables
size_t fused_region_bytes(const sekv_handle* h, FusedParams* P) {
  FusedParams tmp;
  if (!P) P = &tmp;
  size_t need = fused_plan_smem(h, P);
  need = std::max(need, (size_t)kStages * kStageBytes);
  if (h->cfg.k_cap > 0) need = std::max(need, (size_t)h->lay.slot_bytes);
  need = std::max(need, (size_t)kPartStride * 4 * 8);
  return round_up_sz(need, 128);
}

// spans per ROUTE item: their G x dp rows plus q' fit the smallest region
int fused_route_spans(const sekv_handle* h) {
  const int per_span = h->G * h->cfg.route_dim * 2;
  const int cap = (kStages * kStageBytes - h->G * h->cfg.route_dim * 4) / per_span;
  return std::max(8, std::min(64, cap / 8 * 8));
}

int fused_warps(const sekv_handle* h) {
  const size_t region = fused_region_bytes(h, nullptr);
  const size_t budget = 227 * 1024 - 1024;
  return (int)std::min<size_t>(8, budget / region);
}

template <int G>
static cudaError_t launch_fused_g(const FusedParams& P, size_t smem, int grid, int threads, cudaStream_t s, bool pdl) {
  static size_t configured = 0;
  if (smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(fused_layer_kernel<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3(grid); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, fused_layer_kernel<G>, P);
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
  P.partials = (float*)ws(h, h->F.off_partials1);
  P.keys = (uint32_t*)ws(h, h->F.off_keys);
  P.qp = (float*)ws(h, h->F.off_qp);
  P.zdesc = (ZDescG*)ws(h, h->F.off_zdesc) + (size_t)layer * c.max_seqs * c.n_kv_heads * (std::max(c.k_cap, 1) + std::max(c.prefetch, 0));
  P.ctrs = (int32_t*)ws(h, h->F.off_ctrs) + (size_t)layer * h->F.ctrs_per_layer;
  P.plan_counts = (int32_t*)ws(h, h->F.off_plan_counts) + (size_t)layer * c.max_seqs * c.n_kv_heads * 2;
  P.stats = (unsigned long long*)ws(h, h->F.off_stats);
  P.host_arena = h->host_dev;
  {   // trace records of layer l start at record l * (n_items + groups)
    const int64_t stride = (int64_t)h->n_items + (int64_t)h->n_seqs * c.n_kv_heads;
    const int64_t left = h->trace_cap - (int64_t)layer * stride;
    P.trace = (h->trace_buf && left > 0) ? (unsigned long long*)h->trace_buf + 8 * (size_t)layer * stride : nullptr;
    P.trace_cap = left > 0 ? std::min(left, stride) : 0;
  }
  P.mode = mode; P.k = k; P.k_cap = c.k_cap; P.prefetch = std::max(c.prefetch, 0);
  P.kc = std::max(c.k_cap, 1) + std::max(c.prefetch, 0);
  P.BG = h->n_seqs * c.n_kv_heads;
  P.Hq = c.n_q_heads; P.Hkv = c.n_kv_heads; P.dp = c.route_dim; P.ways = c.cache_ways;
  P.mask_words = h->mask_words; P.spans_cap = (int)h->lay.spans_cap; P.m_tot = h->m_tot; P.keys_stride = h->F.keys_per_bg;
  P.out_bf16 = c.out_dtype == SEKV_BF16;
  P.slot_bytes = h->lay.slot_bytes;
  P.ent_head_stride = (size_t)h->lay.rows_cap * kD;
  P.route_head_stride = (size_t)h->lay.spans_cap * c.route_dim;
  P.region_bytes = (int)fused_region_bytes(h, &P);
  P.route_spans = fused_route_spans(h);
  // queues: [QPROJ, ROUTE | SELECT | POOL, ZOOM, COARSE, COMBINE]
  P.pool_end = h->pool_end;
  if ((mode & FM_ROUTE) && (mode & FM_ATTN)) {                  // whole-step launches run the layers in order
    const LayerView nv = layer_view(h, (layer + 1) % c.n_layers);
    P.next_W = (const uint8_t*)nv.W;
    P.next_route = (const uint8_t*)nv.route;
    P.next_W_bytes = (size_t)c.n_q_heads * c.route_dim * kD * 2;
    P.next_route_head_bytes = (size_t)h->m_tot * c.route_dim * 2;
  }
  if (mode == FM_ROUTE) { P.lat_begin = 0; P.lat_end = h->n_lat_items; P.main_end = h->n_lat_items; }
  else if (mode == FM_ATTN) { P.lat_begin = h->select_begin; P.lat_end = h->n_lat_items; P.main_end = h->n_items; }
  else { P.lat_begin = 0; P.lat_end = h->n_lat_items; P.main_end = h->n_items; }
  const size_t smem = (size_t)h->fused_warps * P.region_bytes;
  const int grid = h->fused_grid, threads = 32 * h->fused_warps;
  cudaError_t e;
  switch (h->G) {
    case 1: e = launch_fused_g<1>(P, smem, grid, threads, s, h->use_pdl); break;
    case 2: e = launch_fused_g<2>(P, smem, grid, threads, s, h->use_pdl); break;
    case 3: e = launch_fused_g<3>(P, smem, grid, threads, s, h->use_pdl); break;
    case 4: e = launch_fused_g<4>(P, smem, grid, threads, s, h->use_pdl); break;
    case 5: e = launch_fused_g<5>(P, smem, grid, threads, s, h->use_pdl); break;
    case 6: e = launch_fused_g<6>(P, smem, grid, threads, s, h->use_pdl); break;
    case 7: e = launch_fused_g<7>(P, smem, grid, threads, s, h->use_pdl); break;
    case 8: e = launch_fused_g<8>(P, smem, grid, threads, s, h->use_pdl); break;
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
