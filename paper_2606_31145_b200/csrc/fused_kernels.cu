// The bf16 hot path: ONE persistent kernel per layer-step that runs a1-a7 (Eq. 4, 5, 9, L123,
// L119-121, Eq. 8).  One CTA per SM, kFusedWarps warps, every warp with a private shared-memory region.
//
//   chain (a1-a4), per (sequence, kv head) group bg, by a TEAM of warps of CTA bg % grid, entirely in
//   shared memory (no global round trips between the steps):
//     q' = W q (Eq. 4, tensor cores)  ->  x = q'.K_bar/sqrt(d') + ln|S|, X = max over the group (Eq. 5, GQA;
//     the routing table streams through bulk-copied staging buffers)  ->  top-k by radix select (Eq. 9, cap
//     L123; ties to the lower span id)  ->  residency plan of the device factor cache (LRU), zoom bit-mask,
//     one stamped descriptor per expanded span
//   work items (a5-a7), one warp each, claimed in queue order:
//     POOL    (b, g, rows)   online-softmax partial over full-resolution tokens; no dependency
//     COARSE  (b, g, rows)   partial over the coarse entries (+ln|S|) of the spans that are NOT expanded
//                            (an expanded span's coarse entry is replaced by its tokens); waits
//                            for the group's zoom mask
//     ZOOM    (b, g, 1 span) an expanded span through the factored form (Eq. 8 never materialised); waits for
//                            the span's descriptor; the U factors move by 1-D bulk copies (TMA engine); a demand
//                            miss reads its blob from the pinned-host store over PCIe and keeps it in its slot
//     PREFETCH (b, g, i)     speculative: a candidate of the PREVIOUS layer's plan, pinned host -> cache slot
//     COMBINE (b, h)         log-sum-exp merge of the head's partials -> output (L61)
//
// Waiting items only wait on the teams (which start at t = 0 and wait on nobody) or on items earlier in the
// queue; claims are in queue order and the grid is resident (checked on the host): the wait graph is acyclic.
//
// Tensor cores: G <= 8 query heads per kv head is far below a tcgen05 tile and the path is HBM-bound, so the
// heads are the (padded) rows / columns of warp-level mma.sync.m16n8k16 tiles.
#include <algorithm>

#include "mma_common.cuh"

namespace sekv {

namespace {

constexpr int kStages = 2;                 // ring stages of a rows item (16 rows of K + 16 rows of V each)
constexpr int kStageBytes = 2 * 16 * kD * 2;
constexpr int kFusedWarps = 12;
constexpr int kFusedThreads = 32 * kFusedWarps;
constexpr int kRegionBytes = 19200;        // 12 x 19200 + static < 227 KB

// Monotone map float -> uint32 (larger float => larger key); key 0 is free to mean "not eligible".
__device__ __forceinline__ uint32_t order_key(float x) {
  const uint32_t u = __float_as_uint(x);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

__device__ __forceinline__ void cp_async16(void* dst_smem, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(void* dst_smem, const void* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
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
__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
// 2^x on the special function unit (one MUFU; 2^-inf = 0)
__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// four 8x8 b16 matrices, transposed on the way in (lanes 8j..8j+7 give the row addresses of matrix j)
__device__ __forceinline__ void ldsm_x4_trans(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
// transpose an 8x8 b16 matrix held one row-pair per lane (C-fragment layout -> B-fragment layout)
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t a) {
  uint32_t d;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(d) : "r"(a));
  return d;
}
__device__ __forceinline__ uint4 ld_cg16(const void* p) {       // L2-coherent 16-byte load
  uint4 v;
  asm volatile("ld.global.cg.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}

// header loads of a ZOOM item: the header is in a cache slot (global) or, for a demand miss, staged in shared memory
__device__ __forceinline__ uint4 hdr_ld16(const uint8_t* p, bool in_smem) {
  return in_smem ? *reinterpret_cast<const uint4*>(p) : ld_cg16(p);
}
__device__ __forceinline__ float hdr_ldf(const uint8_t* p, bool in_smem) {
  return in_smem ? *reinterpret_cast<const float*>(p) : __ldcg(reinterpret_cast<const float*>(p));
}

// Counters of a launch (one of two sets per layer, alternating with the layer's launch sequence number: the set a
// launch uses was zeroed during the previous launch of the layer, so nothing is re-armed in the kernel's tail):
// [0] work queue, [1] warps that have read the sequence number, then one word per group: attention items done,
// POOL + COARSE items in the low 16 bits (kEarlyOne), all kinds in the high 16 bits (kAttnOne).
__device__ __forceinline__ int32_t* grp_ctr(int32_t* ctrs, int bg) { return ctrs + 4 + 4 * bg; }
constexpr int kEarlyOne = 0x00010001, kAttnOne = 0x00010000;
// spin (lane 0) until the 16-bit field of the group's counter reaches `target`
__device__ __forceinline__ void wait_field(const int32_t* c, int shift, int target, int lane, unsigned long long* t_mid = nullptr) {
  if (lane == 0) {
    int v;
    for (;;) {
      asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(c) : "memory");
      if (((v >> shift) & 0xFFFF) >= target) break;
      __nanosleep(64);
    }
    asm volatile("fence.acq_rel.gpu;" ::: "memory");
    if (t_mid) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(*t_mid));
  }
  __syncwarp();
}

// trace mark k (0..3) of the current item (lane 0; tm = null when tracing is off)
__device__ __forceinline__ void mark(unsigned long long* tm, int k, int lane) {
  if (tm && lane == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(tm[k]));
}
// Q fragments of the group's heads (rows gid < G; zero rows above): qf[j] = q[gid][8 (t4 + 4 j) .. +7]
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
// The team: warps 0 .. ntw-1 of a CTA, meeting on named barrier 1.  Its tables live at the start of the
// CTA's dynamic shared memory (the regions of the team's own warps), followed by one routing-table staging
// buffer per team warp.
// ---------------------------------------------------------------------------------------------------
struct Team { int tt, ts, lane, tw, ntw; int* scratch; uint8_t* tab; uint8_t* stage; uint64_t* bars; uint32_t ph[2]; };

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

// ---------------------------------------------------------------------------------------------------
// a1 (Eq. 4): q'_h = W_h q_h for one query head on the tensor cores: the rows of W_h are the M dimension
// (16 per tile), the group's queries are the 8 columns, column hl of the result is q'_hl -> shared memory.
// ---------------------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ void qproj_load(const FusedParams& P, int b, int g, int hl, int j0, int lane,
                                           uint32_t (&qf)[4][4], uint4 (&w)[2][2][4], bool with_q = true) {
  const int dp = P.dp, gid = lane >> 2, t4 = lane & 3;
  if (j0 == 0 && with_q) load_q_frags(P.q + ((size_t)b * P.Hq + (size_t)g * G) * kD, G, gid, t4, qf);
  const uint8_t* Wh = (const uint8_t*)P.lv.W + (size_t)(g * G + hl) * dp * (kD * 2) + t4 * 16;
#pragma unroll
  for (int mt = 0; mt < 2; ++mt)
#pragma unroll
    for (int hf = 0; hf < 2; ++hf) {
      const int row = j0 + 16 * mt + 8 * hf + gid;
#pragma unroll
      for (int jj = 0; jj < 4; ++jj)
        w[mt][hf][jj] = row < dp ? ldg16(Wh + (size_t)row * (kD * 2) + jj * 64) : make_uint4(0u, 0u, 0u, 0u);
    }
}
template <int G>
__device__ __forceinline__ void qproj_mma(const FusedParams& P, int hl, int j0, int lane, const uint32_t (&qf)[4][4],
                                          const uint4 (&w)[2][2][4], float* dst) {
  const int dp = P.dp, gid = lane >> 2, t4 = lane & 3;
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

// meta = |S| << 16 | rank_k | rank_v << 8 of the span
// it = way | miss << 31 | no-slot << 30 | way-pending << 29 (a demand miss whose slot the plan has not chosen yet: the
// ZOOM item starts the fetch from the host store and reads `it` from P.zway[j] when it needs the slot);
// j = index of the span in the sorted zoom list (the ZOOM item's partial slot; < 2^15)
__device__ __forceinline__ void write_zdesc(const FusedParams& P, ZDescG* zd, int bg, int g, int span0, int id, uint32_t it,
                                            uint32_t meta, uint32_t epoch, int j = 0) {
  ZDescG d;
  d.src = 0ull; d.bytes = 0u; d.len_rr = 0u; d.way_miss = (it & 0xE0003FFFu) | (((uint32_t)j & 0x7FFFu) << 14); d.id = id;
  d.epoch0 = epoch; d.epoch1 = epoch;
  if (id >= 0) {
    const int gs = span0 + id;
    const int rr = (int)(meta & 0xffffu);
    const int len = (int)(meta >> 16);
    d.len_rr = meta;
    d.bytes = (uint32_t)blob_dims(2, len, rr & 0xff, (rr >> 8) & 0xff).bytes;
    // hits: the cache slot; misses: the device alias of the pinned-host store (the ZOOM item copies the blob into
    // its slot first when it has one)
    const uint8_t* src = (it & 0x80000000u) ? P.host_arena + P.lv.dir_off[(size_t)g * P.spans_cap + gs]
                                            : P.lv.slots + ((size_t)bg * P.ways + (it & 0x3FFFu)) * P.slot_bytes;
    d.src = (unsigned long long)src;
  }
  uint4* o = reinterpret_cast<uint4*>(zd);
  o[0] = make_uint4((uint32_t)d.src, (uint32_t)(d.src >> 32), d.bytes, d.epoch0);
  o[1] = make_uint4(d.len_rr, d.way_miss, (uint32_t)d.id, d.epoch1);
}

struct PlanTables {
  int32_t* sh_ids; int16_t* way_of; int32_t* sh_tag; uint32_t* sh_stamp; int32_t* sh_victim; uint32_t* sh_mask;
  uint32_t* meta;      // [m] |S| << 16 | rank_k | rank_v << 8 of every span of the group
  float* lnl;          // [m] ln|S|
};
__device__ __forceinline__ PlanTables plan_tables(const FusedParams& P, uint8_t* tab) {
  PlanTables t;
  t.sh_ids = reinterpret_cast<int32_t*>(tab + P.sm_ids);
  t.way_of = reinterpret_cast<int16_t*>(tab + P.sm_wayof);
  t.sh_tag = reinterpret_cast<int32_t*>(tab + P.sm_tags);
  t.sh_stamp = reinterpret_cast<uint32_t*>(t.sh_tag + P.ways);
  t.sh_victim = reinterpret_cast<int32_t*>(t.sh_stamp + P.ways);
  t.sh_mask = reinterpret_cast<uint32_t*>(tab + P.sm_mask);
  t.meta = reinterpret_cast<uint32_t*>(tab + P.sm_meta);
  t.lnl = reinterpret_cast<float*>(tab + P.sm_lnl);
  return t;
}

// Tables that need nothing from this step's routing -> shared memory by 4-byte cp.async copies, all in flight at
// once (no register round trip): span meta (the directory word carries |S| and both ranks), ln|S|, cache tags and
// stamps.  The caller commits / waits and runs a team barrier; _scatter then inverts the tags into way_of.
__device__ __forceinline__ void plan_init_fill(const FusedParams& P, const Team& T, const PlanTables& t, int bg, int span0,
                                               int m) {
  const int g = bg % P.Hkv;
  const int32_t* dirw = P.lv.dir_rank + (size_t)g * P.spans_cap + span0;
  const float* lnl = P.cv.ln_len + span0;
#pragma unroll 1
  for (int s = T.tt; s < m; s += T.ts) { cp_async4(t.meta + s, dirw + s); cp_async4(t.lnl + s, lnl + s); t.way_of[s] = (int16_t)-1; }
  if (P.mode & FM_ATTN) {
    const int32_t* tags = P.lv.tags + (size_t)bg * P.ways;
    const uint32_t* stamps = P.lv.stamps + (size_t)bg * P.ways;
#pragma unroll 1
    for (int w = T.tt; w < P.ways; w += T.ts) { cp_async4(t.sh_tag + w, tags + w); cp_async4(t.sh_stamp + w, stamps + w); t.sh_victim[w] = -1; }
  }
  cp_async_commit();
  for (int w = T.tt; w < P.mask_words; w += T.ts) t.sh_mask[w] = 0u;
  if (T.tt == 0) { T.scratch[24] = 0; T.scratch[25] = 0; T.scratch[26] = 0; }   // descriptor positions (plan_team)
}
__device__ __forceinline__ void plan_init_scatter(const FusedParams& P, const Team& T, const PlanTables& t, int m) {
  for (int w = T.tt; w < P.ways; w += T.ts) { const int tg = t.sh_tag[w]; if (tg >= 0 && tg < m) t.way_of[tg] = (int16_t)w; }
}

// ---------------------------------------------------------------------------------------------------
// a1 + a2 + GQA reduce of a3 (Eq. 4, 5, 9) by the team: q' -> shared memory; the G x m rows of the routing
// table of (b, g) stream through the team warps' staging buffers in blocks of P.route_spans spans (cp.async,
// P.route_bufs deep), ordered 32-bit keys -> shared memory.  Fast path (d' = 32, no threshold, no score
// outputs): per head, 16 staged rows are the M dimension of mma tiles, q' (split into bf16 hi + lo, ~16
// bits) the columns.  General path: compact scalar loops.
// ---------------------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ void route_team(const FusedParams& P, Team& T, int bg, uint32_t* keys,
                                           float* sqp, const PlanTables& pt, int* span0_out, int* m_out,
                                           bool pdl_wait, unsigned long long* tm) {
  const int b = bg / P.Hkv, g = bg % P.Hkv, dp = P.dp, lpr = dp >> 3, lane = T.lane;
  // W of this warp's head goes first: it needs nothing but the group index.  With pdl_wait everything up to the
  // query load (static tables only) runs BEFORE the programmatic-dependent-launch wait, i.e. in the tail of the
  // previous layer's kernel; the query -- the one input that depends on the previous layer -- is read after it.
  uint32_t qf[4][4];
  uint4 wq[2][2][4];
  const int my_hl = T.tw;
  if (my_hl < G) qproj_load<G>(P, b, g, my_hl, 0, lane, qf, wq, false);
  const int2 gi = __ldg(P.grp + bg);                             // first span and span count of the group's sequence
  const int span0 = gi.x, m = gi.y;
  *span0_out = span0; *m_out = m;
  const int gid = lane >> 2, t4 = lane & 3;
  const int nsp_blk = P.route_spans, nbuf = P.route_bufs;
  const int nblk = (m + nsp_blk - 1) / nsp_blk;
  const uint8_t* route = (const uint8_t*)P.lv.route;
  const uint32_t buf_bytes = (uint32_t)nsp_blk * G * dp * 2;
  // one 1-D bulk copy per head: the rows of a block are contiguous in the routing table and in the staging buffer
  auto issue = [&](int blk, int buf) {
    __syncwarp();                                              // every lane is done reading this buffer
    if (lane == 0) {
      const int s_lo = blk * nsp_blk, nsp = min(m, s_lo + nsp_blk) - s_lo;
      uint8_t* dst = T.stage + (size_t)buf * buf_bytes;
      const uint32_t hb = (uint32_t)nsp * dp * 2;
      mbar_arrive_expect_tx(&T.bars[buf], hb * G);
#pragma unroll 1
      for (int hl = 0; hl < G; ++hl)
        bulk_g2s(dst + (size_t)hl * hb, route + ((size_t)(g * G + hl) * P.route_head_stride + (size_t)(span0 + s_lo) * dp) * 2,
                 hb, &T.bars[buf]);
    }
  };
  int blk = T.tw, buf = 0;
  if (blk < nblk) issue(blk, 0);
  if (nbuf == 2 && blk + T.ntw < nblk) issue(blk + T.ntw, 1);
  plan_init_fill(P, T, pt, bg, span0, m);                       // independent of the routing: its loads overlap
  int* sel = T.scratch + 16;                                     // [2..4] eligible keys / min key / max key
  if (T.tt == 0) { sel[2] = 0; sel[3] = -1; sel[4] = 0; sel[5] = 0; sel[6] = 0; }
  {
    uint32_t* hist = reinterpret_cast<uint32_t*>(T.tab + P.sm_hist);     // one histogram per radix pass of the select
    for (int i = T.tt; i < 4 * 256; i += T.ts) hist[i] = 0u;
  }
  if (pdl_wait) asm volatile("griddepcontrol.wait;" ::: "memory");
  if (my_hl < G) {
    load_q_frags(P.q + ((size_t)b * P.Hq + (size_t)g * G) * kD, G, lane >> 2, lane & 3, qf);
    qproj_mma<G>(P, my_hl, 0, lane, qf, wq, sqp + my_hl * dp);
    for (int j0 = 32; j0 < dp; j0 += 32) {                       // d' = 64: the second half of W_h
      qproj_load<G>(P, b, g, my_hl, j0, lane, qf, wq);
      qproj_mma<G>(P, my_hl, j0, lane, qf, wq, sqp + my_hl * dp);
    }
  }
  for (int hl = my_hl + T.ntw; hl < G; hl += T.ntw)              // (teams with fewer warps than heads)
    for (int j0 = 0; j0 < dp; j0 += 32) {
      qproj_load<G>(P, b, g, hl, j0, lane, qf, wq);
      qproj_mma<G>(P, hl, j0, lane, qf, wq, sqp + hl * dp);
    }
  cp_async_wait<0>();
  team_bar(T);                                                   // q' of the group and the plan tables are in shared memory
  if (P.mode & FM_ATTN) plan_init_scatter(P, T, pt, m);
  int ne = 0;
  uint32_t kmin = 0xFFFFFFFFu, kmax = 0u;
  const float inv_sqrt_dp = rsqrtf((float)dp);
  const bool fast = dp == 32 && P.tau == nullptr && P.logits_out == nullptr && P.alpha_out == nullptr;
  uint32_t bh[4] = {0u, 0u, 0u, 0u}, bl[4] = {0u, 0u, 0u, 0u};
  if (fast && gid < G) {
    const float4 v0 = *reinterpret_cast<const float4*>(sqp + gid * 32 + 8 * t4);
    const float4 v1 = *reinterpret_cast<const float4*>(sqp + gid * 32 + 8 * t4 + 4);
    split_bf16(v0.x * inv_sqrt_dp, v0.y * inv_sqrt_dp, bh[0], bl[0]);
    split_bf16(v0.z * inv_sqrt_dp, v0.w * inv_sqrt_dp, bh[1], bl[1]);
    split_bf16(v1.x * inv_sqrt_dp, v1.y * inv_sqrt_dp, bh[2], bl[2]);
    split_bf16(v1.z * inv_sqrt_dp, v1.w * inv_sqrt_dp, bh[3], bl[3]);
  }
  for (; blk < nblk; blk += T.ntw) {
    mbar_wait(&T.bars[buf], T.ph[buf]);
    T.ph[buf] ^= 1u;
    const int s_lo = blk * nsp_blk, nsp = min(m, s_lo + nsp_blk) - s_lo;
    const uint8_t* src = T.stage + (size_t)buf * buf_bytes;
    if (fast) {
#pragma unroll 1
      for (int s0 = 0; s0 < nsp; s0 += 16) {
        float Xa = -INFINITY, Xb = -INFINITY;                      // spans s0 + gid and s0 + gid + 8
#pragma unroll
        for (int hl = 0; hl < G; ++hl) {
          const uint8_t* ra = src + ((size_t)hl * nsp + s0 + gid) * 64 + t4 * 16;
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
        if (t4 < 2 && s < nsp) {
          const uint32_t k = order_key(((t4 & 1) ? Xb : Xa) + pt.lnl[s_lo + s]);
          keys[s_lo + s] = k;
          ++ne; kmin = min(kmin, k); kmax = max(kmax, k);
        }
      }
    } else {
      for (int s = lane; s < nsp; s += 32) {
        const float lnl = pt.lnl[s_lo + s];
        float X = -INFINITY;
        bool elig = (P.tau == nullptr);
#pragma unroll 1
        for (int hl = 0; hl < G; ++hl) {
          const uint4* row = reinterpret_cast<const uint4*>(src + ((size_t)hl * nsp + s) * dp * 2);
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
          if (P.logits_out) P.logits_out[(size_t)h * P.m_tot + span0 + s_lo + s] = x;
          if (P.alpha_out) P.alpha_out[(size_t)h * P.m_tot + span0 + s_lo + s] = a;
          if (P.tau != nullptr && a > P.tau[h]) elig = true;       // Eq. 9
          X = fmaxf(X, x);
        }
        const uint32_t k = elig ? order_key(X) : 0u;
        keys[s_lo + s] = k;
        if (k != 0u) { ++ne; kmin = min(kmin, k); kmax = max(kmax, k); }
      }
    }
    const int nb = blk + nbuf * T.ntw;                           // the block that reuses this buffer
    if (nb < nblk) issue(nb, buf);
    if (nbuf == 2) buf ^= 1;
  }
  // eligible keys, smallest and largest key of the group (what the radix select starts from)
  ne = warp_sum_i(ne);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    kmin = min(kmin, __shfl_xor_sync(0xffffffffu, kmin, o));
    kmax = max(kmax, __shfl_xor_sync(0xffffffffu, kmax, o));
  }
  if (lane == 0 && ne > 0) {
    atomicAdd(&sel[2], ne);
    atomicMin(reinterpret_cast<unsigned int*>(&sel[3]), kmin);
    atomicMax(reinterpret_cast<unsigned int*>(&sel[4]), kmax);
  }
  team_bar(T);                                                   // the keys of the group are complete
  mark(tm, 0, T.tt);
}

// The zoom mask is all the COARSE items wait for.  It is published as self-validating (bits, step stamp) pairs --
// 8-byte stores that the COARSE items poll; no flag, no fence.
__device__ __forceinline__ void publish_mask(const FusedParams& P, const Team& T, const PlanTables& t, int bg, uint32_t epoch) {
  uint2* gmask = P.zmask2 + (size_t)bg * P.mask_words;
  for (int w = T.tt; w < P.mask_words; w += T.ts) gmask[w] = make_uint2(t.sh_mask[w], epoch);
}

// a4: residency plan of (b, g).  The device factor cache of a (layer, sequence, kv head) is `ways` slots with
// a tag (span id) and a stamp (step of last use).  The first n_zoom entries of sh_ids are this step's zoom
// set: resident ones are hits, the others are demand misses and take the least-recently-used slots not
// needed by this step.  Entries n_zoom .. n_cand-1 are prefetch candidates (the next-best spans by routing
// score): the non-resident ones get a slot too and are copied by the side-stream prefetch kernel after
// this layer's kernel.  Also: zoom bit-mask for the COARSE items (an expanded span's coarse entry is
// replaced by its tokens), de-duplication of caller-supplied ids, one descriptor per
// expanded span for the ZOOM items, statistics.
__device__ __forceinline__ void plan_team(const FusedParams& P, const Team& T_in, const PlanTables& t, int bg, int span0,
                                          int m, int n_zoom, int n_cand, bool dedupe, uint32_t epoch,
                                          bool mask_done, bool solo_tail, unsigned long long* tm = nullptr) {
  Team T = T_in;
  const int g = bg % P.Hkv, ways = P.ways;
  int32_t* tags = P.lv.tags + (size_t)bg * ways;
  uint32_t* stamps = P.lv.stamps + (size_t)bg * ways;
  uint32_t* items = P.lv.items + (size_t)bg * P.kc;
  int32_t* item_span = P.lv.item_span + (size_t)bg * P.kc;
  ZDescG* zd = P.zdesc + (size_t)bg * P.kc;
  const uint32_t cur = epoch;
  // Descriptor positions of the zoom set: ZOOM item i of the group polls zd[i], and the items are claimed in
  // that order.  Demand misses (slowest: their blob crosses PCIe) take the first positions; hits and "none"
  // entries fill the positions from the back.  Every list index j < K gets exactly one descriptor, which
  // carries j: the partial of span j always lands in slot j, so the merge order -- and the output bits -- do not
  // depend on which position (or warp) a span went to.  Prefetch candidate c is zd[kcap1 + c].
  const int K = min(P.k_cap, m);
  int* pos_hit = T.scratch + 24; int* pos_miss = T.scratch + 25;
  int n_hit = 0, n_miss = 0, n_pf = 0, n_pf_slot = 0;
  unsigned long long bytes_algo = 0, bytes_demand = 0, bytes_pf = 0;
  // pass 1: validate / de-duplicate, zoom mask, residency lookup
  for (int j = T.tt; j < max(n_cand, K); j += T.ts) {
    if (j >= n_zoom && j < K)                                  // list index past the zoom set: "none", done at once
      write_zdesc(P, zd + (K - 1 - atomicAdd(pos_hit, 1)), bg, g, span0, -1, 0u, 0u, epoch, j);
    if (j >= n_cand) continue;
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
      if (zoom) {
        bytes_algo += (unsigned long long)(rk + rv) * (len + kD) * 2 + 4ull * (rk + rv);
        if (way >= 0) ++n_hit;
        else { ++n_miss; bytes_demand += blob_dims(2, len, rk, rv).bytes; }
      } else if (way < 0) ++n_pf;
    }
    t.sh_ids[j] = id;
    item_span[j] = id;
    items[j] = (way >= 0) ? (uint32_t)way : 0xFFFFFFFFu;
    // hits publish their descriptor at once: the ZOOM items poll it and start while the misses are still
    // being given slots; a resident prefetch candidate needs no copy
    if (zoom && (way >= 0 || id < 0))
      write_zdesc(P, zd + (K - 1 - atomicAdd(pos_hit, 1)), bg, g, span0, id, (uint32_t)max(way, 0), meta, epoch, j);
    // ... and so do the demand misses, before their slot is known: their blob crosses PCIe (the longest pole of the
    // layer at a few misses per step), and the fetch needs the slot only when the first bytes have arrived
    if (zoom && id >= 0 && way < 0)
      write_zdesc(P, zd + atomicAdd(pos_miss, 1), bg, g, span0, id, 0xA0000000u, meta, epoch, j);
  }
  int n_need;
  team_excl_scan(T, n_miss + n_pf, &n_need);                   // (its barriers also publish pass 1 to the team)
  n_need = min(n_need, ways);
  if (!mask_done) publish_mask(P, T, t, bg, epoch);
  if (T.tt == 0) { P.plan_counts[2 * bg] = n_zoom; P.plan_counts[2 * bg + 1] = n_cand; }
  // statistics of pass 1 (every warp its own share)
  n_hit = warp_sum_i(n_hit); n_miss = warp_sum_i(n_miss);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    bytes_algo += __shfl_xor_sync(0xffffffffu, bytes_algo, o);
    bytes_demand += __shfl_xor_sync(0xffffffffu, bytes_demand, o);
  }
  if (T.lane == 0) {
    if (n_hit) atomicAdd(&P.stats[ST_HITS], (unsigned long long)n_hit);
    if (n_miss) atomicAdd(&P.stats[ST_MISSES], (unsigned long long)n_miss);
    if (n_hit + n_miss) {
      atomicAdd(&P.stats[ST_ZOOMED], (unsigned long long)(n_hit + n_miss));
      atomicAdd(&P.stats[ST_SKIPPED], (unsigned long long)(n_hit + n_miss));
    }
    if (bytes_algo) atomicAdd(&P.stats[ST_FACTOR_ALGO], bytes_algo);
    if (bytes_demand) atomicAdd(&P.stats[ST_H2D], bytes_demand);
  }
  // The mask and the descriptors of the hits are out: what is left (slots for the misses, the cache tables) is
  // little and serial.  With solo_tail the team's warps 1.. leave here for the work queue and warp 0 finishes
  // alone (the tables sit in its own region).
  if (solo_tail) {
    team_bar(T);
    if (T.tw != 0) {
      // On the way out: pull the resident blobs of the zoom set towards L2 (one prefetch per 128-byte line, fire and
      // forget).  The ZOOM items run a few microseconds from now, after the COARSE items, and HBM is idle meanwhile.
      for (int j = T.tw - 1; j < n_zoom; j += T.ntw - 1) {
        const int id = t.sh_ids[j];
        if (id < 0) continue;
        const int way = t.way_of[id];
        if (way < 0) continue;
        const uint32_t meta = t.meta[id];
        const uint32_t lines = (uint32_t)(blob_dims(2, (int)(meta >> 16), meta & 0xff, (meta >> 8) & 0xff).bytes >> 7);
        const uint8_t* base = P.lv.slots + ((size_t)bg * ways + way) * P.slot_bytes;
        for (uint32_t i = T.lane; i < lines; i += 32) asm volatile("prefetch.global.L2 [%0];" ::"l"(base + ((size_t)i << 7)));
      }
      return;
    }
    T.tt = T.lane; T.ts = 32; T.ntw = 1;
  }
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
        if (j >= n_zoom) {                                     // a prefetch candidate that will be copied
          const uint32_t meta = t.meta[id];
          ++n_pf_slot;
          bytes_pf += blob_dims(2, (int)(meta >> 16), meta & 0xff, (meta >> 8) & 0xff).bytes;
        }
      } else {
        it = 0xC0000000u;                                      // no free slot: fetch, do not keep
      }
      items[j] = it;
    }
    miss_base += tot;
    if (miss && j < n_zoom) P.zway[(size_t)bg * P.kc + j] = make_uint2(it, epoch);      // the slot of demand miss j (self-validating pair)
  }
  team_bar(T);
  for (int w = T.tt; w < ways; w += T.ts) { tags[w] = t.sh_tag[w]; stamps[w] = t.sh_stamp[w]; }
  // statistics of pass 2
  n_pf_slot = warp_sum_i(n_pf_slot);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) bytes_pf += __shfl_xor_sync(0xffffffffu, bytes_pf, o);
  if (T.lane == 0) {
    if (bytes_pf) atomicAdd(&P.stats[ST_PF_BYTES], bytes_pf);
    if (n_pf_slot) atomicAdd(&P.stats[ST_PREFETCHED], (unsigned long long)n_pf_slot);
  }
}

// ---------------------------------------------------------------------------------------------------
// a3 (Eq. 9, cap L123): top-n_cand of the group's m keys (shared memory).  A radix select (8 bits per pass,
// shared-memory histograms, starting at the highest bit in which the eligible keys differ) finds the
// n_cand-th largest key T; keys > T are taken, keys == T are taken in increasing span id until the count is
// met (ties to the lower id); the winners are then ranked by (key descending, id ascending).
// Returns cnt (zoom set) and n_cand (zoom set + prefetch candidates); ids in t.sh_ids.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void select_team(const FusedParams& P, const Team& T, const PlanTables& t, const uint32_t* keys,
                                            int m, int* cnt_out, int* ncand_out, unsigned long long* tm) {
  uint32_t* hist = reinterpret_cast<uint32_t*>(T.tab + P.sm_hist);
  unsigned long long* cand = reinterpret_cast<unsigned long long*>(T.tab + P.sm_cand);
  int* sel = T.scratch + 16;     // [0] digit, [1] keys above it, [2..4] ne / kmin / kmax, [5] keys == T, [6] slot
  const int n_elig = sel[2];
  const uint32_t kmin = (uint32_t)sel[3], kmax = (uint32_t)sel[4];
  int cnt = P.k < 0 ? n_elig : min(P.k, n_elig);
  cnt = min(cnt, P.k_cap);
  int n_cand = cnt;
  if (P.k >= 0 && (P.mode & FM_ATTN)) n_cand = min(min(cnt + P.prefetch, n_elig), P.kc);
  uint32_t Tk = 0u;           // threshold key
  int need = 0;               // keys == Tk to take
  const bool partial = n_cand != 0 && n_cand < n_elig;
  if (partial) {
    // the eligible keys agree on every bit above the highest bit in which kmin and kmax differ: the passes
    // start there (float keys of one binade share 9 bits: a pass over them would pile every key -- and
    // every shared-memory atomic -- into one bin)
    const int hb = 31 - __clz((int)((kmin ^ kmax) | 1u));
    const int top = min(24, max(0, hb - 7));                    // first digit = bits [top, top + 8)
    uint32_t maskb = (top + 8 >= 32) ? 0u : ~((1u << (top + 8)) - 1u);
    uint32_t prefix = kmax & maskb;
    need = n_cand;
    uint32_t* hp = hist;
#pragma unroll 1
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
      if (sel[5] == need) break;        // every key of this bin is taken: the lower bits need not be resolved
    }
    Tk = prefix;                        // (after an early exit: the smallest possible key of the bin)
  }
  mark(tm, 1, T.tt);
  // winners: every eligible key (n_cand == n_elig), or the keys > T plus `need` keys == T.  When more keys
  // equal T than are taken, those are taken in increasing span id (ties to the lower id): the rank of a tied
  // key among its equals is counted directly (ties at the cut are rare and few).
  const bool cut_ties = partial && sel[5] != need;
  if (n_cand != 0)
    for (int i = T.tt; i < m; i += T.ts) {
      const uint32_t k = keys[i];
      bool take = partial ? (k > Tk || (k == Tk && !cut_ties)) : (k != 0u);
      if (k == 0u) take = false;
      if (partial && cut_ties && k == Tk) {
        int before = 0;
        for (int j = 0; j < i; ++j) before += (keys[j] == Tk);
        take = before < need;
      }
      if (take) {
        const int pos = atomicAdd(&sel[6], 1);
        if (pos < P.kc) cand[pos] = ((unsigned long long)k << 32) | (unsigned long long)(0xFFFFFFFFu - (uint32_t)i);
      }
    }
  team_bar(T);
  // rank by (key descending, id ascending): the composite 64-bit values are distinct
  for (int j = T.tt; j < n_cand; j += T.ts) {
    const unsigned long long mine = cand[j];
    int r = 0;
    for (int i = 0; i < n_cand; ++i) r += (cand[i] > mine);
    t.sh_ids[r] = (int32_t)(0xFFFFFFFFu - (uint32_t)(mine & 0xFFFFFFFFull));
  }
  team_bar(T);
  mark(tm, 2, T.tt);
  *cnt_out = cnt; *ncand_out = n_cand;
}

// ---------------------------------------------------------------------------------------------------
// The whole chain a1-a4 of group bg by the team.
// ---------------------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ void chain_group(const FusedParams& P, Team& T, int bg, uint32_t& epoch, bool pdl_wait,
                                            bool solo_tail, unsigned long long* tm) {
  const PlanTables t = plan_tables(P, T.tab);
  uint32_t* keys = reinterpret_cast<uint32_t*>(T.tab + P.sm_keys);
  float* sqp = reinterpret_cast<float*>(T.tab + P.sm_qp);
  int span0, m;
  if (P.mode & FM_ROUTE) {
    route_team<G>(P, T, bg, keys, sqp, t, &span0, &m, pdl_wait, tm);
    int cnt, n_cand;
    select_team(P, T, t, keys, m, &cnt, &n_cand, tm);
    int32_t* my_ids = P.ids + (size_t)bg * max(P.k_cap, 1);
    for (int j = T.tt; j < P.k_cap; j += T.ts) my_ids[j] = j < cnt ? t.sh_ids[j] : -1;
    if (T.tt == 0) P.count[bg] = cnt;
    if (P.mode & FM_ATTN) {
      // the zoom set is known: its mask goes out first (routed ids are valid and distinct)
      for (int j = T.tt; j < cnt; j += T.ts) atomicOr(&t.sh_mask[t.sh_ids[j] >> 5], 1u << (t.sh_ids[j] & 31));
      team_bar(T);
      publish_mask(P, T, t, bg, epoch);
      mark(tm, 3, T.tt);
      plan_team(P, T, t, bg, span0, m, cnt, n_cand, false, epoch, true, solo_tail, tm);
    }
  } else {
    // caller-supplied zoom set (sekv_decode_attn)
    const int2 gi = __ldg(P.grp + bg);
    span0 = gi.x; m = gi.y;
    plan_init_fill(P, T, t, bg, span0, m);
    int cnt = 0;
    if (P.ids != nullptr && P.count != nullptr) cnt = max(0, min(P.count[bg], P.k_cap));
    const int32_t* src = P.ids + (size_t)bg * max(P.k_cap, 1);
    for (int j = T.tt; j < cnt; j += T.ts) t.sh_ids[j] = src[j];
    cp_async_wait<0>();
    team_bar(T);
    plan_init_scatter(P, T, t, m);
    team_bar(T);
    plan_team(P, T, t, bg, span0, m, cnt, cnt, true, epoch, false, solo_tail);
  }
}

// one partial record (m2, l, pad, pad, o[128]) per head
__device__ __forceinline__ float* part_ptr(const FusedParams& P, const Item& I, int hl) {
  return P.partials + ((size_t)I.pbase + (size_t)hl * I.np + I.part) * kPartStride;
}
// Lane (gid, t4) holds head gid's running max m_run and its share of l_run, and the O^T accumulators
// of[md][2 hi + c] = O[head 2 t4 + c][dim 16 md + 8 hi + gid].
template <int G>
__device__ __forceinline__ void store_partial(const FusedParams& P, const Item& I, int lane, float m_run, float l_run,
                                              const float (&of)[8][4]) {
  const int gid = lane >> 2, t4 = lane & 3;
  l_run = quad_sum(l_run);
  if (gid < G && t4 == 0) {
    float* pp = part_ptr(P, I, gid);
    pp[0] = m_run; pp[1] = l_run;
  }
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    const int hh = 2 * t4 + c;
    if (hh < G) {
      float* o = part_ptr(P, I, hh) + 4 + gid;
#pragma unroll
      for (int md = 0; md < 8; ++md) { o[16 * md] = of[md][c]; o[16 * md + 8] = of[md][2 + c]; }
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// a5: rows [I.a, I.b) of the entry table of (b, g): pool tokens (logit = q.K/sqrt(d)) and unexpanded coarse
// entries (logit = q.k_bar/sqrt(d) + ln|S|, value v_bar).  16-row tiles of K and V
// stream through a kStages-deep cp.async ring in the warp's region.  Shared-memory layout of a stage:
// K rows then V rows, 256 bytes per row; 16-byte chunk c of row r is stored at chunk c ^ ((r & 1) << 2)
// (K) or c ^ (r & 7) (V): both fragment access patterns below are bank-conflict free.
//   QK^T : lane (gid = lane/4, t4 = lane%4) reads chunk (t4 + 4j) of the K row of token gid; its four
//          words are the (b0,b1) pairs of two k-steps; Q is loaded the same way (the contraction index
//          may be permuted consistently on both operands).
//   P V  : computed transposed, O^T = V^T P^T (M = 16 dims, N = 8 heads, K = 16 tokens): the A fragments
//          come from ldmatrix.trans over the V rows, the C fragment of S IS the B fragment of P^T.
//          P (fp32) is split into bf16 hi + lo parts and multiplied twice, so probabilities carry ~16 bits.
// ---------------------------------------------------------------------------------------------------
// The item after a POOL item is claimed while the POOL item runs: lane 0 issues the atomic when kAheadTiles tiles are
// left, the result is read (and the next descriptor loaded) two tiles later, so neither round trip is exposed.  Not
// earlier: a claim binds the item to this warp, and the warps that finish their POOL rows first should get the items
// at the head of the queue (measured: -0.7 us per layer-step against claiming when the item starts).
constexpr int kAheadTiles = 6;
struct Ahead { int pending, nidx, n_static; bool on, done, issued; Item nxt; };
__device__ __forceinline__ Item load_item(const Item* p);
__device__ __forceinline__ void ahead_resolve(const FusedParams& P, Ahead& a) {
  if (a.on && !a.done) {
    a.nidx = a.n_static + __shfl_sync(0xffffffffu, a.pending, 0);
    if (a.nidx < P.main_end) a.nxt = load_item(P.items + a.nidx);
    a.done = true;
  }
}

// One 16-row K/V tile of a rows item -> ring stage t % kStages (cp.async).  Chunk idx = lane + 32 i of a 16 x 256-byte
// tile is row r = 2 i + (lane >> 4), 16-byte chunk c = lane & 15: global offsets are contiguous and both swizzles are
// per-lane constants plus compile-time terms in i.
__device__ __forceinline__ void rows_fill(const FusedParams& P, const Item& I, uint8_t* region, int lane, int t) {
  const int g = I.bg % P.Hkv, row_begin = I.a, row_end = I.b;
  const uint8_t* Kb = (const uint8_t*)P.lv.ent_k + ((size_t)g * P.ent_head_stride + (size_t)I.row0 * kD) * 2;
  const uint8_t* Vb = (const uint8_t*)P.lv.ent_v + ((size_t)g * P.ent_head_stride + (size_t)I.row0 * kD) * 2;
  const int lr = lane >> 4, lc = lane & 15;
  const uint32_t dk0 = (uint32_t)(lr * 256 + ((lc ^ (lr << 2)) << 4));
  const uint32_t dv0 = (uint32_t)(lr * 256);
  const uint32_t lcx = (uint32_t)(lc ^ lr);
  uint8_t* Ks = region + (t % kStages) * kStageBytes;
  uint8_t* Vs = Ks + 16 * kD * 2;
  const int r0 = row_begin + t * 16;
  if (r0 + 16 <= row_end) {                                   // full tile: no clamping
    const size_t src = (size_t)r0 * (kD * 2) + lane * 16;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      cp_async16(Ks + dk0 + 512 * i, Kb + src + 512 * i);
      cp_async16(Vs + dv0 + 512 * i + ((lcx ^ ((2 * i) & 7)) << 4), Vb + src + 512 * i);
    }
  } else {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int r = 2 * i + lr;
      const size_t src = (size_t)min(r0 + r, row_end - 1) * (kD * 2) + lc * 16;
      cp_async16(Ks + dk0 + 512 * i, Kb + src);
      cp_async16(Vs + dv0 + 512 * i + ((lcx ^ ((2 * i) & 7)) << 4), Vb + src);
    }
  }
}
// the first kStages tiles of a rows item (static tables: may run before the programmatic-dependent-launch wait)
__device__ __forceinline__ void rows_prefill(const FusedParams& P, const Item& I, uint8_t* region, int lane) {
  const int ntiles = (I.b - I.a + 15) >> 4;
#pragma unroll
  for (int t = 0; t < kStages; ++t) {
    if (t < ntiles) rows_fill(P, I, region, lane, t);
    cp_async_commit();
  }
}

template <int G>
__device__ __forceinline__ void rows_item(const FusedParams& P, const Item& I, uint8_t* region, int lane, uint32_t epoch,
                                          int32_t* ctrs, Ahead& ah, bool prefilled, unsigned long long* tm) {
  const int bg = I.bg, b = bg / P.Hkv, g = bg % P.Hkv;
  const int gid = lane >> 2, t4 = lane & 3;
  const int A = I.A, row_begin = I.a, row_end = I.b;
  const float scale2 = rsqrtf((float)kD) * kLog2e;
  const int ntiles = (row_end - row_begin + 15) >> 4;
  if (!prefilled) rows_prefill(P, I, region, lane);
  uint32_t qf[4][4];                                           // (before the COARSE item's poll: its latency overlaps the wait)
  load_q_frags(P.q + ((size_t)b * P.Hq + (size_t)g * G) * kD, G, gid, t4, qf);

  // biases of a COARSE item: lane L holds rows row_begin + L and row_begin + 32 + L (ln|S| in the base-2 domain;
  // -inf for an expanded span, whose coarse entry is replaced by its tokens, and for rows past the item)
  float bias_reg[2] = {0.f, 0.f};
  if (I.kind == IT_COARSE) {
    const uint2* gmask = P.zmask2 + (size_t)bg * P.mask_words;
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int row = row_begin + 32 * u + lane;
      float bias = -INFINITY;
      if (row < row_end) {
        const int sp = row - A;
        const float lnl2 = P.cv.ln_len[I.span0 + sp] * kLog2e;       // (before the poll: independent of the mask)
        bool zoomed = false;
        if (P.k_cap > 0) {                        // poll the mask word until it carries this launch's stamp
          uint2 w;
          for (;;) {
            asm volatile("ld.relaxed.gpu.global.v2.u32 {%0,%1}, [%2];" : "=r"(w.x), "=r"(w.y) : "l"(gmask + (sp >> 5)) : "memory");
            if (w.y == epoch) break;
            __nanosleep(64);
          }
          zoomed = (w.x >> (sp & 31)) & 1u;
        }
        if (!zoomed) bias = lnl2;
      }
      bias_reg[u] = bias;
    }
    __syncwarp();
    mark(tm, 0, lane);
  }
  float m_run = -INFINITY, l_run = 0.f;
  float of[8][4];
#pragma unroll
  for (int md = 0; md < 8; ++md) { of[md][0] = 0.f; of[md][1] = 0.f; of[md][2] = 0.f; of[md][3] = 0.f; }
  // ldmatrix.x4.trans row addresses of this lane: matrix j = lane >> 3 is tokens 8 (j >> 1) .. +7, 16-byte chunk
  // 2 md + (j & 1) of the V rows
  const int lj = lane >> 3, lrow = lane & 7;
  const uint32_t v_tok_off = (uint32_t)((lrow + 8 * (lj >> 1)) * 256);
  const uint32_t v_cx = (uint32_t)((lj & 1) ^ lrow);

  const int t_claim = max(0, ntiles - kAheadTiles), t_res = min(ntiles - 1, t_claim + 2);
  for (int t = 0; t < ntiles; ++t) {
    if (ah.on && t == t_claim) {
      if (lane == 0) ah.pending = atomicAdd(ctrs, 1);
      ah.issued = true;
    }
    cp_async_wait<kStages - 1>();
    __syncwarp();
    const uint8_t* Ks = region + (t % kStages) * kStageBytes;
    const uint32_t Vs = smem_u32(Ks + 16 * kD * 2) + v_tok_off;
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
          z[nt][e] = (bias == -INFINITY) ? -INFINITY : fmaf(sacc[nt][e], scale2, bias);
        }
    }
    const float mx = quad_max(fmaxf(fmaxf(z[0][0], z[0][1]), fmaxf(z[1][0], z[1][1])));
    const float m_new = fmaxf(m_run, mx);
    const float m_safe = (m_new == -INFINITY) ? 0.f : m_new;
    if (__any_sync(0xffffffffu, m_new > m_run)) {
      const float corr = ex2(m_run - m_safe);           // this lane's head is gid
      l_run *= corr;
      const float ca = __shfl_sync(0xffffffffu, corr, 8 * t4);       // head 2*t4
      const float cb = __shfl_sync(0xffffffffu, corr, 8 * t4 + 4);   // head 2*t4+1
#pragma unroll
      for (int md = 0; md < 8; ++md) { of[md][0] *= ca; of[md][1] *= cb; of[md][2] *= ca; of[md][3] *= cb; }
    }
    m_run = m_new;
    const float p00 = ex2(z[0][0] - m_safe), p01 = ex2(z[0][1] - m_safe);
    const float p10 = ex2(z[1][0] - m_safe), p11 = ex2(z[1][1] - m_safe);
    l_run += (p00 + p01) + (p10 + p11);
    uint32_t b0h, b0l, b1h, b1l;          // P^T fragments: n = head gid, k = tokens 2*t4+e (b0) and 8+2*t4+e (b1)
    split_bf16(p00, p01, b0h, b0l);
    split_bf16(p10, p11, b1h, b1l);
#pragma unroll
    for (int md = 0; md < 8; ++md) {
      uint32_t a0, a1, a2, a3;
      ldsm_x4_trans(Vs + ((v_cx ^ (2 * md)) << 4), a0, a1, a2, a3);
      mma16816_full(of[md], a0, a1, a2, a3, b0h, b1h);
      mma16816_full(of[md], a0, a1, a2, a3, b0l, b1l);
    }
    __syncwarp();                                      // every lane is done with this stage
    if (t + kStages < ntiles) rows_fill(P, I, region, lane, t + kStages);
    cp_async_commit();
    if (ah.issued && t == t_res) ahead_resolve(P, ah);
  }
  if (ah.on && !ah.issued) { if (lane == 0) ah.pending = atomicAdd(ctrs, 1); ah.issued = true; }     // (an item without tiles)
  cp_async_wait<0>();
  ahead_resolve(P, ah);
  store_partial<G>(P, I, lane, m_run, l_run, of);
  __syncwarp();
  if (lane == 0) red_add_release(grp_ctr(ctrs, bg), kEarlyOne);
}

// lane 0 starts a 1-D bulk copy into the warp's region (completion on `bar`); callers wait with mbar_wait
__device__ __forceinline__ void region_fetch_start(uint8_t* region, const void* src, uint32_t bytes, uint64_t* bar, int lane) {
  __syncwarp();                                    // every lane is done with the region's previous contents
  if (lane == 0) {
    fence_proxy_async();                           // (shared::cta) generic writes to the region before the async-proxy write
    mbar_arrive_expect_tx(bar, bytes);
    bulk_g2s(region, src, bytes, bar);
  }
}
__device__ __forceinline__ void region_fetch(uint8_t* region, const void* src, uint32_t bytes, uint64_t* bar,
                                             uint32_t& phase, int lane) {
  region_fetch_start(region, src, bytes, bar, lane);
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
// a6: one expanded span through the factored form (Eq. 8 never materialised).  Every operand is read in its
// mma fragment order (sekv_internal.cuh): Vt_K, sigma and V_V straight from global memory (L2), the
// per-token factors U_K, U_V from the warp's region, where they arrive by 1-D bulk copies in windows of as
// many 16-token chunks as the region holds.
//   c   = sigma_K o (Vt_K q) * log2e/sqrt(d)       heads x rank           (A: q,       B: Vt_K)
//   S   = c U_K^T                                   heads x tokens         (A: c,       B: U_K)
//   p   = 2^(S - m)
//   y^T = U_V^T p^T                                 rank x heads           (A: U_V^T,   B: p^T = C fragment of S)
//   O^T += V_V (sigma_V o y)^T                      dims x heads           (A: V_V,     B: y^T through movmatrix)
// NK: compile-time bound on the 16-wide k-steps over the key and value ranks (1 or 4).
// ---------------------------------------------------------------------------------------------------
template <int G, int NK>
__device__ __forceinline__ void zoom_span(const FusedParams& P, const uint8_t* __restrict__ blob, const uint8_t* hdr,
                                          bool hdr_smem, int len, int nks, int nvs, uint8_t* region, uint32_t cap_bytes,
                                          uint64_t* bar, uint32_t& phase, int lane,
                                          const uint32_t (&qf)[4][4], float& M, float& L, float (&of)[8][4],
                                          uint8_t* wb, bool wb_regs, uint64_t* hbar, uint32_t* hphase, uint32_t hdr_bytes,
                                          unsigned long long* tm) {
  // blob: where the chunk windows come from (cache slot, or the pinned-host copy of a demand miss); hdr: the header
  // (= blob, or a copy staged in shared memory); region / cap_bytes: where the windows go.
  // wb: null, or the cache slot a demand miss is kept in: the chunk windows are written to it by bulk copies out
  // of the region (and, with wb_regs, the header pieces this warp holds in registers by plain stores).
  // (M, L, of) are OUTPUTS: the span's own online-softmax partial (one span per ZOOM item)
  const int gid = lane >> 2, t4 = lane & 3;
  const size_t off_sv = (size_t)nks * 64, off_vtk = (size_t)(nks + nvs) * 64;
  const size_t off_vv = off_vtk + (size_t)nks * 4096, off_ch = off_vv + (size_t)nvs * 4096;
  const uint32_t chunk_bytes = (uint32_t)(nks + nvs) * 512u;
  const int nchunks = (len + 15) >> 4;
  // (windows hold a multiple of CH chunks, so the iterations group the same chunks whatever the window size:
  // a span gives the same bits from a cache slot and from the host store)
  constexpr int CH = NK == 1 ? 4 : 2;
  const int fit = (int)(cap_bytes / chunk_bytes);
  const int win = max(1, min(nchunks, fit >= CH ? fit / CH * CH : fit));
  const float scale2 = rsqrtf((float)kD) * kLog2e;
  region_fetch_start(region, blob + off_ch, (uint32_t)min(win, nchunks) * chunk_bytes, bar, lane);
  if (hbar != nullptr) {                               // demand miss: the staged header (in flight together with the window)
    mbar_wait(hbar, *hphase);
    *hphase ^= 1u;
    if (wb && lane == 0) { bulk_s2g(wb, hdr, hdr_bytes); bulk_commit(); }
  }
  // V_V is needed last: pull it towards L2 now
  if (NK != 1 && !hdr_smem)
    for (int i = lane; i < nvs * 32; i += 32) asm volatile("prefetch.global.L2 [%0];" ::"l"(hdr + off_vv + (size_t)i * 128));
  // 1. c
  uint32_t ckh[NK][2], ckl[NK][2];
#pragma unroll
  for (int ks = 0; ks < NK; ++ks) {
    ckh[ks][0] = ckh[ks][1] = ckl[ks][0] = ckl[ks][1] = 0u;
    if (ks < nks) {
      uint4 kv[2][4];
#pragma unroll
      for (int u = 0; u < 2; ++u)
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) kv[u][jj] = hdr_ld16(hdr + off_vtk + (size_t)(((ks * 2 + u) * 4 + jj) * 512 + lane * 16), hdr_smem);
      const uint4 skr = hdr_ld16(hdr + (size_t)ks * 64 + t4 * 16, hdr_smem);      // sigma_K[16 ks + 4 t4 .. + 3]
      if (wb && wb_regs) {
#pragma unroll
        for (int u = 0; u < 2; ++u)
#pragma unroll
          for (int jj = 0; jj < 4; ++jj)
            *reinterpret_cast<uint4*>(wb + off_vtk + (size_t)(((ks * 2 + u) * 4 + jj) * 512 + lane * 16)) = kv[u][jj];
        if (gid == 0) *reinterpret_cast<uint4*>(wb + (size_t)ks * 64 + t4 * 16) = skr;
      }
      const float sk[4] = {__uint_as_float(skr.x), __uint_as_float(skr.y), __uint_as_float(skr.z), __uint_as_float(skr.w)};
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        float cf[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
          mma16816(cf, qf[jj][0], qf[jj][1], kv[u][jj].x, kv[u][jj].y);
          mma16816(cf, qf[jj][2], qf[jj][3], kv[u][jj].z, kv[u][jj].w);
        }
        // columns 2*t4+e of n-tile u are rank index 16 ks + 4 t4 + 2 u + e
        split_bf16(cf[0] * (sk[2 * u] * scale2), cf[1] * (sk[2 * u + 1] * scale2), ckh[ks][u], ckl[ks][u]);
      }
    }
  }
  mark(tm, 1, lane);
  // V_V and sigma_V are needed last: with one k-step (rank <= 16) their loads are issued now and land during the
  // token loop (32 registers); otherwise they are loaded in the epilogue
  uint4 vv0[8];
  float sv0_lo = 0.f, sv0_hi = 0.f;
  if (NK == 1) {
#pragma unroll
    for (int md = 0; md < 8; ++md) vv0[md] = hdr_ld16(hdr + off_vv + (size_t)(md * 512 + lane * 16), hdr_smem);
    sv0_lo = hdr_ldf(hdr + off_sv + 4 * gid, hdr_smem);
    sv0_hi = hdr_ldf(hdr + off_sv + 4 * (8 + gid), hdr_smem);
    if (wb && wb_regs) {
#pragma unroll
      for (int md = 0; md < 8; ++md) *reinterpret_cast<uint4*>(wb + off_vv + (size_t)(md * 512 + lane * 16)) = vv0[md];
      if (t4 == 0) {
        reinterpret_cast<float*>(wb + off_sv)[gid] = sv0_lo;
        reinterpret_cast<float*>(wb + off_sv)[8 + gid] = sv0_hi;
      }
    }
  }
  // 2. the token chunks, CH per iteration: their logits are independent, one running-max update serves all of
  // them; y accumulates in two independent sets (even / odd chunks) to halve the dependent mma chain
  float m_s = -INFINITY, l_s = 0.f;
  float yf[2][NK][4];
#pragma unroll
  for (int a2 = 0; a2 < 2; ++a2)
#pragma unroll
    for (int n = 0; n < NK; ++n) { yf[a2][n][0] = yf[a2][n][1] = yf[a2][n][2] = yf[a2][n][3] = 0.f; }
  for (int w0 = 0; w0 < nchunks; w0 += win) {
    const int nwc = min(win, nchunks - w0);
    mbar_wait(bar, phase);
    phase ^= 1u;
    if (wb && lane == 0) {                             // keep the window: region -> slot (async, read-only on the region)
      bulk_s2g(wb + off_ch + (size_t)w0 * chunk_bytes, region, (uint32_t)nwc * chunk_bytes);
      bulk_commit();
    }
    for (int c = 0; c < nwc; c += CH) {
      const int nact = min(CH, nwc - c);
      const uint8_t* ch = region + (size_t)c * chunk_bytes + lane * 16;
      float sacc[CH][2][4];
#pragma unroll
      for (int cc = 0; cc < CH; ++cc) {
#pragma unroll
        for (int nt = 0; nt < 2; ++nt) sacc[cc][nt][0] = sacc[cc][nt][1] = sacc[cc][nt][2] = sacc[cc][nt][3] = 0.f;
        if (cc < nact) {
#pragma unroll
          for (int ks = 0; ks < NK; ++ks) {
            if (ks < nks) {
              const uint4 bv = *reinterpret_cast<const uint4*>(ch + (size_t)cc * chunk_bytes + ks * 512);
              mma16816(sacc[cc][0], ckh[ks][0], ckh[ks][1], bv.x, bv.y);
              mma16816(sacc[cc][1], ckh[ks][0], ckh[ks][1], bv.z, bv.w);
              mma16816(sacc[cc][0], ckl[ks][0], ckl[ks][1], bv.x, bv.y);
              mma16816(sacc[cc][1], ckl[ks][0], ckl[ks][1], bv.z, bv.w);
            }
          }
        }
      }
      // this lane: head gid, tokens 16 (w0 + c + cc) + 8 nt + 2 t4 + e
      const int tok0 = 16 * (w0 + c);
      if (tok0 + 16 * CH > len || nact < CH) {         // warp-uniform: only the tail needs masking
#pragma unroll
        for (int cc = 0; cc < CH; ++cc)
#pragma unroll
          for (int nt = 0; nt < 2; ++nt)
#pragma unroll
            for (int e = 0; e < 2; ++e)
              if (tok0 + 16 * cc + 8 * nt + 2 * t4 + e >= len || cc >= nact) sacc[cc][nt][e] = -INFINITY;
      }
      float mx = -INFINITY;
#pragma unroll
      for (int cc = 0; cc < CH; ++cc)
        mx = fmaxf(mx, fmaxf(fmaxf(sacc[cc][0][0], sacc[cc][0][1]), fmaxf(sacc[cc][1][0], sacc[cc][1][1])));
      mx = quad_max(mx);
      const float m_new = fmaxf(m_s, mx);
      const float m_safe = (m_new == -INFINITY) ? 0.f : m_new;
      if (__any_sync(0xffffffffu, m_new > m_s)) {
        const float corr = ex2(m_s - m_safe);
        l_s *= corr;
        const float ca = __shfl_sync(0xffffffffu, corr, 8 * t4), cb = __shfl_sync(0xffffffffu, corr, 8 * t4 + 4);
#pragma unroll
        for (int a2 = 0; a2 < 2; ++a2)
#pragma unroll
          for (int n = 0; n < NK; ++n) { yf[a2][n][0] *= ca; yf[a2][n][1] *= cb; yf[a2][n][2] *= ca; yf[a2][n][3] *= cb; }
      }
      m_s = m_new;
#pragma unroll
      for (int cc = 0; cc < CH; ++cc) {
        if (cc < nact) {
          const float p00 = ex2(sacc[cc][0][0] - m_safe), p01 = ex2(sacc[cc][0][1] - m_safe);
          const float p10 = ex2(sacc[cc][1][0] - m_safe), p11 = ex2(sacc[cc][1][1] - m_safe);
          l_s += (p00 + p01) + (p10 + p11);
          uint32_t b0h, b0l, b1h, b1l;      // P^T fragments: n = head gid, k = tokens 2 t4 + e (b0), 8 + 2 t4 + e (b1)
          split_bf16(p00, p01, b0h, b0l);
          split_bf16(p10, p11, b1h, b1l);
#pragma unroll
          for (int mv = 0; mv < NK; ++mv) {
            if (mv < nvs) {
              const uint4 av = *reinterpret_cast<const uint4*>(ch + (size_t)cc * chunk_bytes + (nks + mv) * 512);
              mma16816_full(yf[cc & 1][mv], av.x, av.y, av.z, av.w, b0h, b1h);
              mma16816_full(yf[cc & 1][mv], av.x, av.y, av.z, av.w, b0l, b1l);
            }
          }
        }
      }
    }
    if (w0 + win < nchunks) {
      if (wb && lane == 0) bulk_wait_read_all();        // the write-back has read the region
      region_fetch_start(region, blob + off_ch + (size_t)(w0 + win) * chunk_bytes,
                         (uint32_t)min(win, nchunks - w0 - win) * chunk_bytes, bar, lane);
    }
  }
  if (wb && lane == 0) bulk_wait_all();
  mark(tm, 2, lane);
  // 3. O^T = V_V (sigma_V o y)^T
  M = m_s;
  L = l_s;
#pragma unroll
  for (int md = 0; md < 8; ++md) { of[md][0] = 0.f; of[md][1] = 0.f; of[md][2] = 0.f; of[md][3] = 0.f; }
#pragma unroll
  for (int kv = 0; kv < NK; ++kv) {
    if (kv < nvs) {
      // y[2 hi + c] is y^T[i = 16 kv + 8 hi + gid][head 2 t4 + c]
      const float y0 = yf[0][kv][0] + yf[1][kv][0], y1 = yf[0][kv][1] + yf[1][kv][1];
      const float y2 = yf[0][kv][2] + yf[1][kv][2], y3 = yf[0][kv][3] + yf[1][kv][3];
      const float sv_lo = NK == 1 ? sv0_lo : hdr_ldf(hdr + off_sv + 4 * (16 * kv + gid), hdr_smem);
      const float sv_hi = NK == 1 ? sv0_hi : hdr_ldf(hdr + off_sv + 4 * (16 * kv + 8 + gid), hdr_smem);
      if (NK != 1 && wb && wb_regs && t4 == 0) {
        reinterpret_cast<float*>(wb + off_sv)[16 * kv + gid] = sv_lo;
        reinterpret_cast<float*>(wb + off_sv)[16 * kv + 8 + gid] = sv_hi;
      }
      uint32_t h0, l0, h1, l1;
      split_bf16(y0 * sv_lo, y1 * sv_lo, h0, l0);
      split_bf16(y2 * sv_hi, y3 * sv_hi, h1, l1);
      const uint32_t b0h = movmatrix_trans(h0), b1h = movmatrix_trans(h1);
      const uint32_t b0l = movmatrix_trans(l0), b1l = movmatrix_trans(l1);
#pragma unroll
      for (int md = 0; md < 8; ++md) {
        const uint4 av = NK == 1 ? vv0[md] : hdr_ld16(hdr + off_vv + (size_t)((kv * 8 + md) * 512 + lane * 16), hdr_smem);
        if (NK != 1 && wb && wb_regs) *reinterpret_cast<uint4*>(wb + off_vv + (size_t)((kv * 8 + md) * 512 + lane * 16)) = av;
        mma16816_full(of[md], av.x, av.y, av.z, av.w, b0h, b1h);
        mma16816_full(of[md], av.x, av.y, av.z, av.w, b0l, b1l);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// a4 + a6: plan items [I.a, I.b) of (b, g), one expanded span after the other.  A demand miss is first
// copied from the pinned-host store (device-mapped, over PCIe) into the cache slot the plan gave it and then
// read from there like a hit; without a free slot it is read straight from the host store.
// ---------------------------------------------------------------------------------------------------
template <int G>
__device__ __forceinline__ void zoom_item(const FusedParams& P, const Item& I, uint8_t* region, uint64_t* bar,
                                          uint32_t& phase, uint32_t& phase1, int lane, uint32_t epoch, int32_t* ctrs,
                                          unsigned long long* tm) {
  const int bg = I.bg, b = bg / P.Hkv, g = bg % P.Hkv;
  const int gid = lane >> 2, t4 = lane & 3;
  uint32_t qf[4][4];
  load_q_frags(P.q + ((size_t)b * P.Hq + (size_t)g * G) * kD, G, gid, t4, qf);
  // ONE span per ZOOM item (the plan stamps every descriptor of the schedule; id -1 = none)
  float M = -INFINITY, L = 0.f;
  float of[8][4];
  const ZDescG d = poll_zdesc(P.zdesc + (size_t)bg * P.kc + I.a, epoch);
  mark(tm, 0, lane);
  if (d.id >= 0) {
    const uint8_t* blob = reinterpret_cast<const uint8_t*>(d.src);
    const int len = (int)(d.len_rr >> 16);
    const int nks = max(1, ((int)(d.len_rr & 0xff) + 15) >> 4), nvs = max(1, ((int)((d.len_rr >> 8) & 0xff) + 15) >> 4);
    // Demand miss: the blob is read from the pinned-host store over PCIe by the bulk-copy engine only (plain loads
    // of host memory turn into many 32-byte PCIe reads): first the header into the front of the region (and on into
    // the slot, when the plan gave it one), then the chunk windows behind it, each kept in the slot on the way.
    const bool miss = (d.way_miss & 0x80000000u) != 0u;
    const uint32_t hdr_bytes = (uint32_t)(nks + nvs) * (64u + 4096u), chunk_bytes = (uint32_t)(nks + nvs) * 512u;
    const uint8_t* hdr = blob;
    uint8_t* cbase = region;
    uint32_t cap = (uint32_t)P.region_bytes;
    bool hdr_smem = false;
    uint64_t* hbar = nullptr;
    if (miss && hdr_bytes + chunk_bytes <= (uint32_t)P.region_bytes) {
      __syncwarp();
      if (lane == 0) {                                 // header -> front of the region, on the warp's second barrier
        mbar_arrive_expect_tx(bar + 1, hdr_bytes);
        bulk_g2s(region, blob, hdr_bytes, bar + 1);
      }
      hbar = bar + 1;
      hdr = region; hdr_smem = true;
      cbase = region + hdr_bytes; cap = (uint32_t)P.region_bytes - hdr_bytes;
    }
    // the slot of a demand miss (the header is already on its way): chosen by the plan a little after the descriptor
    uint8_t* wb = nullptr;
    if (miss) {
      uint32_t it = d.way_miss;
      if (it & 0x20000000u) {
        const uint2* zw = P.zway + (size_t)bg * P.kc + ((d.way_miss >> 14) & 0x7FFFu);
        uint2 w;
        for (;;) {
          asm volatile("ld.relaxed.gpu.global.v2.u32 {%0,%1}, [%2];" : "=r"(w.x), "=r"(w.y) : "l"(zw) : "memory");
          if (w.y == epoch) break;
          __nanosleep(64);
        }
        it = w.x;
      }
      if ((it & 0xC0000000u) == 0x80000000u) wb = P.lv.slots + ((size_t)bg * P.ways + (it & 0x3FFFu)) * P.slot_bytes;
    }
    const bool wb_regs = wb != nullptr && !hdr_smem;
    if (nks <= 1 && nvs <= 1)
      zoom_span<G, 1>(P, blob, hdr, hdr_smem, len, 1, 1, cbase, cap, bar, phase, lane, qf, M, L, of, wb, wb_regs, hbar, &phase1, hdr_bytes, tm);
    else
      zoom_span<G, 4>(P, blob, hdr, hdr_smem, len, nks, nvs, cbase, cap, bar, phase, lane, qf, M, L, of, wb, wb_regs, hbar, &phase1, hdr_bytes, tm);
  } else {
#pragma unroll
    for (int n = 0; n < 8; ++n) { of[n][0] = of[n][1] = of[n][2] = of[n][3] = 0.f; }
  }
  mark(tm, 3, lane);
  Item Ij = I;                                                   // the partial of list index j goes to slot j
  Ij.part = I.part - I.a + (int)((d.way_miss >> 14) & 0x7FFFu);
  store_partial<G>(P, Ij, lane, M, L, of);
  __syncwarp();
  if (lane == 0) red_add_release(grp_ctr(ctrs, bg), kAttnOne);
}

// ---------------------------------------------------------------------------------------------------
// a4, speculative prefetch: candidate I.a of group (b, g) of the PREVIOUS layer of this step -- one of the
// next-best spans by routing score that was not resident and that the previous layer's plan gave a slot -- is
// copied pinned host -> slot by the bulk-copy engine, bounced through the warp's region.  The previous layer's
// kernel is complete (plain loads of its plan), its cache is next read one step later, and the copy has this
// whole kernel to cross PCIe: it is on nobody's critical path.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void prefetch_item(const FusedParams& P, const Item& I, uint8_t* region, uint64_t* bar,
                                              uint32_t& phase, int lane) {
  const int bg = I.bg, g = bg % P.Hkv;
  const int j = P.pf_plan_counts[2 * bg] + I.a;
  if (j >= P.pf_plan_counts[2 * bg + 1]) return;
  const int id = P.pf_lv.item_span[(size_t)bg * P.kc + j];
  const uint32_t it = P.pf_lv.items[(size_t)bg * P.kc + j];
  if (id < 0 || (it & 0xC0000000u) != 0x80000000u) return;
  const int gs = I.span0 + id;
  const uint32_t rr = (uint32_t)P.pf_lv.dir_rank[(size_t)g * P.spans_cap + gs];   // |S| << 16 | r_V << 8 | r_K
  const uint32_t bytes = (uint32_t)blob_dims(2, (int)(rr >> 16), rr & 0xff, (rr >> 8) & 0xff).bytes;
  const uint8_t* src = P.host_arena + P.pf_lv.dir_off[(size_t)g * P.spans_cap + gs];
  uint8_t* dst = P.pf_lv.slots + ((size_t)bg * P.ways + (it & 0x3FFFu)) * P.slot_bytes;
  __syncwarp();
  if (lane == 0) {
    const uint32_t piece = (uint32_t)P.region_bytes;
    for (uint32_t o = 0; o < bytes; o += piece) {
      const uint32_t n = min(piece, bytes - o);
      mbar_arrive_expect_tx(bar, n);
      bulk_g2s(region, src + o, n, bar);
      mbar_wait(bar, phase);
      phase ^= 1u;
      bulk_s2g(dst + o, region, n);
      bulk_commit();
      bulk_wait_read_all();                          // the region may be overwritten by the next piece
    }
    bulk_wait_all();
  }
  phase = __shfl_sync(0xffffffffu, phase, 0);
}

// ---------------------------------------------------------------------------------------------------
// a7 (L61): log-sum-exp merge of the np partials of one query head -> out, lse.  The head's records are
// contiguous; they move into the warp's region by bulk copies and are reduced from shared memory.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void combine_item(const FusedParams& P, const Item& I, uint8_t* region, uint64_t* bar,
                                             uint32_t& phase, int lane, int32_t* ctrs, unsigned long long* tm) {
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
  wait_field(grp_ctr(ctrs, bg), 0, n_pool, lane, nullptr);
  bool second = false;
  for (int p0 = 0; p0 < np; p0 += cap) {
    if (!second && p0 >= n_pool) { wait_field(grp_ctr(ctrs, bg), 16, np, lane, tm); second = true; }
    const int n = min(cap, (second ? np : n_pool) - p0);
    region_fetch(region, src + (size_t)p0 * kPartStride, (uint32_t)(n * kPartStride * 4), bar, phase, lane);
    float mc = -INFINITY;
    for (int p = lane; p < n; p += 32) mc = fmaxf(mc, rec[p * kPartStride]);
    mc = warp_max(mc);
    const float Mn = fmaxf(M, mc);
    const float safe = (Mn == -INFINITY) ? 0.f : Mn;
    const float c_old = ex2(M - safe);
    // weights in parallel (lane p), kept in the record's pad word; L by a warp reduction
    float lsum = 0.f;
    for (int p = lane; p < n; p += 32) {
      const float mp = rec[p * kPartStride];
      const float w = (mp == -INFINITY) ? 0.f : ex2(mp - safe);
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
  if (!second) wait_field(grp_ctr(ctrs, bg), 16, np, lane, tm);  // (no ZOOM partials at all)
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
__global__ void __launch_bounds__(kFusedThreads, 1) fused_layer_kernel(const __grid_constant__ FusedParams P) {
  extern __shared__ __align__(128) uint8_t dsm[];
  __shared__ uint64_t bars[kFusedWarps][2];
  __shared__ unsigned long long tmid_s[kFusedWarps * 4];
  __shared__ int team_scratch[32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nw = blockDim.x >> 5;
  // Programmatic dependent launch: the next layer's grid may be scheduled as soon as this one's CTAs leave
  // their SMs (its CTAs then sit in the wait below), which hides the launch latency between the dependent
  // kernels of a step; everything this kernel touches is ordered after the previous grid by the wait.
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  uint8_t* region = dsm + (size_t)warp * P.region_bytes;
  uint64_t* bar = &bars[warp][0];
  if (lane == 0) {
    mbar_init(&bars[warp][0], 1);
    mbar_init(&bars[warp][1], 1);
    mbar_fence_init();
  }
  __syncwarp();
  uint32_t phase = 0u, phase1 = 0u;                   // parities of the warp's two barriers
  unsigned long long* tm = P.trace ? &tmid_s[warp * 4] : nullptr;

  // The chain of group bg runs on the team (warps 0 .. team_warps-1) of CTA bg % grid, starting at t = 0.  All
  // other warps take their first work item statically (no claim latency at the start) and claim from there on.
  // Whatever needs only static tables runs BEFORE the dependency wait, i.e. while the previous layer's kernel
  // drains: the first K/V tiles of a POOL item, and (P.hoist) the chain's tables, routing blocks and W.  The
  // query -- the one input that depends on the previous layer -- is read after the wait.
  const int ntw = P.team_warps;
  const int n_chain_cta = P.has_chain ? min(P.BG, (int)gridDim.x) : 0;
  const bool chain_cta = (int)blockIdx.x < n_chain_cta;
  const bool is_team = chain_cta && warp < ntw;
  uint32_t epoch = 0u;
  int idx = -1;
  Item first;
  bool prefilled = false, pf_done = false;
  if (!is_team) {
    const int b = (int)blockIdx.x;
    idx = chain_cta ? b * (nw - ntw) + (warp - ntw) : n_chain_cta * (nw - ntw) + (b - n_chain_cta) * nw + warp;
    if (idx < P.main_end) {
      first = load_item(P.items + idx);
      if (first.kind == IT_POOL) { rows_prefill(P, first, region, lane); prefilled = true; }
      // P.pf_early: the prefetch candidates this launch copies are those of the layer TWO launches back.  That launch is
      // complete whenever a CTA of this one runs: the grid holds one CTA per SM, so this CTA got its SM from a CTA of
      // the previous launch that has exited, i.e. that passed its own dependency wait.  The copy therefore runs here,
      // BEFORE the wait, while this SM has nothing else to do: a copy from the host store in flight slows the SM's
      // other memory traffic down (a pool item next to one took 16 us instead of 10, profiles/r02_item_trace.md).
      if (first.kind == IT_PREFETCH && P.pf_early) {
        if (P.pf_plan_counts != nullptr) prefetch_item(P, first, region, bar, phase, lane);
        pf_done = true;
      }
    }
  }
  // The layer's step stamp and launch sequence number (which picks the counter set) are only written by launches
  // of THIS layer.  With P.hoist the kernel before this one on the stream is the previous layer's of the same
  // step, so both are settled and can be read before the wait; otherwise after it.
  if (!P.hoist) asm volatile("griddepcontrol.wait;" ::: "memory");
  epoch = *reinterpret_cast<volatile const uint32_t*>(P.lv.layer_step) + 1u;
  const uint32_t seq = *reinterpret_cast<volatile const uint32_t*>(P.ctrs);
  int32_t* ctrs = P.ctrs + 4 + (seq & 1u) * P.ctrs_set;
  if (P.hoist && !is_team) asm volatile("griddepcontrol.wait;" ::: "memory");
  if (is_team) {
    Team T;
    T.tt = tid; T.ts = ntw * 32; T.lane = lane; T.tw = warp; T.ntw = ntw; T.scratch = team_scratch;
    T.tab = dsm; T.stage = dsm + P.sm_stage + (size_t)warp * P.stage_bytes;
    T.bars = &bars[warp][0]; T.ph[0] = 0u; T.ph[1] = 0u;
    bool pdl_wait = P.hoist != 0;
    for (int bg = (int)blockIdx.x; bg < P.BG; bg += (int)gridDim.x) {
      unsigned long long t0 = 0ull;
      if (P.trace) { t0 = globaltimer_ns(); if (lane == 0) { tm[0] = t0; tm[1] = t0; tm[2] = t0; tm[3] = t0; } }
      // the last group of this CTA: once its mask and hit descriptors are out, warps 1.. go on to the work queue
      // (only when the team's tables fit warp 0's own region: the released warps reuse theirs)
      const bool solo_tail = (P.mode & FM_ATTN) && bg + (int)gridDim.x >= P.BG && P.sm_stage <= P.region_bytes;
      chain_group<G>(P, T, bg, epoch, pdl_wait, solo_tail, tm);
      pdl_wait = false;
      if (solo_tail && warp != 0) break;
      const int rec = P.main_end + bg;                         // trace record after the queue items
      if (P.trace && tid == 0 && rec < P.trace_cap) {
        unsigned long long* r = P.trace + 8 * (size_t)rec;
        r[0] = (unsigned long long)(uint32_t)IT_SELECT | ((unsigned long long)(uint32_t)bg << 32);
        r[1] = (unsigned long long)blockIdx.x;
        r[2] = t0; r[3] = globaltimer_ns();
        r[4] = tm[0]; r[5] = tm[1]; r[6] = tm[2]; r[7] = tm[3];
      }
      if (!solo_tail) team_bar(T);                             // the tables are free for the next group
    }
    phase = T.ph[0]; phase1 = T.ph[1];                         // the items go on with this warp's barriers
  }
  // this warp has read the layer's sequence number and step stamp (both are advanced by one thread at the end of
  // the launch, once every warp of the grid has said so here)
  __syncwarp();
  if (lane == 0) asm volatile("red.relaxed.gpu.global.add.s32 [%0], %1;" ::"l"(ctrs + 1), "r"(1) : "memory");
  if (blockIdx.x == gridDim.x - 1) {                             // the other set: for the next launch of this layer
    int32_t* other = P.ctrs + 4 + ((seq + 1u) & 1u) * P.ctrs_set;
    for (int i = tid; i < P.ctrs_set; i += blockDim.x) other[i] = 0;
  }
  const int n_static = n_chain_cta * (nw - ntw) + ((int)gridDim.x - n_chain_cta) * nw;
  auto claim = [&]() -> int {
    int i = 0;
    if (lane == 0) i = n_static + atomicAdd(ctrs, 1);
    return __shfl_sync(0xffffffffu, i, 0);
  };
  if (is_team) idx = claim();
  if (idx < P.main_end) {
    // Claims run ahead only through POOL items (dependency-free: the claimed item does not wait long behind them).
    // Any other item is claimed when the warp is free to run it: a claim binds the item to this warp, and an item
    // bound behind a COARSE or ZOOM item that is waiting for its chain starts later than it would on a free warp
    // (measured: -0.7 us per layer-step at 100% hits against claiming ahead through COARSE items too).
    Item cur = is_team ? load_item(P.items + idx) : first;
    for (;;) {
      Ahead ah;
      ah.on = cur.kind == IT_POOL; ah.done = false; ah.issued = false; ah.n_static = n_static; ah.pending = 0; ah.nidx = P.main_end;
      unsigned long long t0 = 0ull;
      const int cur_idx = idx;
      if (P.trace) { t0 = globaltimer_ns(); if (lane == 0) { tm[0] = t0; tm[1] = t0; tm[2] = t0; tm[3] = t0; } }
      switch (cur.kind) {
        case IT_POOL:
        case IT_COARSE: rows_item<G>(P, cur, region, lane, epoch, ctrs, ah, prefilled, tm); prefilled = false; break;
        case IT_ZOOM: zoom_item<G>(P, cur, region, bar, phase, phase1, lane, epoch, ctrs, tm); break;
        case IT_PREFETCH: if (P.pf_plan_counts != nullptr && !pf_done) prefetch_item(P, cur, region, bar, phase, lane); pf_done = false; break;
        default: combine_item(P, cur, region, bar, phase, lane, ctrs, tm); break;
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
      if (ah.on) {
        idx = ah.nidx;
        if (idx >= P.main_end) break;
        cur = ah.nxt;
      } else {
        idx = claim();
        if (idx >= P.main_end) break;
        cur = load_item(P.items + idx);
      }
    }
  }
  // an exiting warp has nothing left to claim, and the tail of the kernel is latency-bound: pull the tables
  // that head the next layer's dependency chain (W, routing summaries) into L2 while HBM is idle
  if (P.next_W != nullptr) {
    const int total_w = (int)gridDim.x * nw, gw = (int)blockIdx.x * nw + warp;
    const size_t w_lines = P.next_W_bytes >> 7, r_lines = P.next_route_head_bytes >> 7;
    for (size_t i = (size_t)gw * 32 + lane; i < w_lines; i += (size_t)total_w * 32)
      asm volatile("prefetch.global.L2 [%0];" ::"l"(P.next_W + (i << 7)));
    for (size_t i = (size_t)gw * 32 + lane; i < r_lines * P.Hq; i += (size_t)total_w * 32) {
      const size_t h = i / r_lines, li = i - h * r_lines;
      asm volatile("prefetch.global.L2 [%0];" ::"l"(P.next_route + h * P.route_head_stride * 2 + (li << 7)));
    }
  }
  // Nothing is re-armed here and no CTA waits for another one on the way out.  One thread advances the layer's
  // sequence number and step stamp once every CTA has read them (they did at their start; the count is a check).
  if (blockIdx.x == 0 && tid == 0) {
    int v;
    for (;;) {
      asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(ctrs + 1) : "memory");
      if (v >= (int)(gridDim.x * (blockDim.x >> 5))) break;
      __nanosleep(64);
    }
    *reinterpret_cast<volatile uint32_t*>(P.ctrs) = seq + 1u;
    if (P.mode & FM_ATTN) {
      *P.lv.layer_step = epoch;
      atomicAdd(&P.stats[ST_LAYER_STEPS], 1ull);
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// The same copies as prefetch_item by a kernel of their own, for the cases in which no following layer kernel
// can carry them: a one-layer model, or a caller that reads the last layer's cache before the next step.
// One warp per candidate; lane 0 drives bulk copies through a shared-memory bounce buffer.
// ---------------------------------------------------------------------------------------------------
constexpr uint32_t kBounceBytes = 32768;
__global__ void __launch_bounds__(32) prefetch_kernel(CsrView cv, LayerView lv, const int32_t* __restrict__ plan_counts,
                                                      int kc, int Hkv, int ways, int spans_cap, int64_t slot_bytes,
                                                      const uint8_t* __restrict__ host_arena) {
  extern __shared__ __align__(128) uint8_t buf[];
  __shared__ uint64_t bar;
  const int bg = blockIdx.y, g = bg % Hkv;
  const int j = plan_counts[2 * bg] + blockIdx.x;
  if (j >= plan_counts[2 * bg + 1]) return;
  const int id = lv.item_span[(size_t)bg * kc + j];
  const uint32_t it = lv.items[(size_t)bg * kc + j];
  if (id < 0 || (it & 0xC0000000u) != 0x80000000u) return;
  if (threadIdx.x == 0) {
    const int gs = cv.seq_span_off[bg / Hkv] + id;
    const uint32_t rr = (uint32_t)lv.dir_rank[(size_t)g * spans_cap + gs];
    const uint32_t bytes = (uint32_t)blob_dims(2, (int)(rr >> 16), rr & 0xff, (rr >> 8) & 0xff).bytes;
    const uint8_t* src = host_arena + lv.dir_off[(size_t)g * spans_cap + gs];
    uint8_t* dst = lv.slots + ((size_t)bg * ways + (it & 0x3FFFu)) * slot_bytes;
    mbar_init(&bar, 1);
    mbar_fence_init();
    uint32_t ph = 0u;
    for (uint32_t o = 0; o < bytes; o += kBounceBytes) {
      const uint32_t n = min(kBounceBytes, bytes - o);
      mbar_arrive_expect_tx(&bar, n);
      bulk_g2s(buf, src + o, n, &bar);
      mbar_wait(&bar, ph);
      ph ^= 1u;
      bulk_s2g(dst + o, buf, n);
      bulk_commit();
      bulk_wait_read_all();
    }
    bulk_wait_all();
  }
}

}  // namespace

// ---------------------------------------------------------------------------------------------------
// host side: shared-memory plan, launchers
// ---------------------------------------------------------------------------------------------------
static int pow2_ceil(int x) { int p = 1; while (p < x) p <<= 1; return p; }

// byte offsets of the team's tables at the start of the CTA's dynamic shared memory; returns their size
static size_t fused_team_tables(const sekv_handle* h, FusedParams* P) {
  const sekv_config& c = h->cfg;
  const int kc = std::max(c.k_cap, 1) + std::max(c.prefetch, 0);
  const int mm = std::max(h->max_m, 1);
  size_t o = 0;
  P->sm_keys = (int)o; o += (size_t)round_up(mm, 4) * 4;
  o = round_up_sz(o, 16); P->sm_hist = (int)o; o += 4 * 256 * 4;
  o = round_up_sz(o, 16); P->sm_cand = (int)o; o += (size_t)pow2_ceil(std::max(kc, 64)) * 8;
  o = round_up_sz(o, 16); P->sm_ids = (int)o; o += (size_t)kc * 4;
  o = round_up_sz(o, 16); P->sm_wayof = (int)o; o += (size_t)round_up(mm, 8) * 2;
  o = round_up_sz(o, 16); P->sm_tags = (int)o; o += (size_t)c.cache_ways * 12;
  o = round_up_sz(o, 16); P->sm_mask = (int)o; o += (size_t)h->mask_words * 4;
  o = round_up_sz(o, 16); P->sm_meta = (int)o; o += (size_t)round_up(mm, 4) * 4;
  o = round_up_sz(o, 16); P->sm_lnl = (int)o; o += (size_t)round_up(mm, 4) * 4;
  o = round_up_sz(o, 16); P->sm_qp = (int)o; o += (size_t)h->G * c.route_dim * 4;
  return round_up_sz(o, 128);
}

// Shared-memory geometry of the fused kernel for the segmented batch: per-warp regions, the team's tables and
// routing-table staging buffers.  Returns false (with a reason) when the batch does not fit the kernel.
bool fused_geometry(const sekv_handle* h, FusedParams* P, std::string* why) {
  const sekv_config& c = h->cfg;
  FusedParams tmp;
  if (!P) P = &tmp;
  const int BG = h->n_seqs * c.n_kv_heads;
  P->region_bytes = kRegionBytes;
  P->team_warps = BG <= h->num_sms ? kFusedWarps : kFusedWarps / 2;
  const size_t tables = fused_team_tables(h, P);
  const size_t team_bytes = (size_t)P->team_warps * kRegionBytes;
  const int per_span = h->G * c.route_dim * 2;
  if (tables + (size_t)P->team_warps * 8 * per_span > team_bytes) {
    if (why) *why = "select / plan tables of the longest sequence do not fit the team's shared memory";
    return false;
  }
  P->sm_stage = (int)tables;
  P->stage_bytes = (int)((team_bytes - tables) / P->team_warps / 128 * 128);
  // spans per routing block: a multiple of 16 (mma tiles of the fast path), two buffers when they fit
  const int fit = P->stage_bytes / per_span;
  if (fit >= 32) { P->route_bufs = 2; P->route_spans = std::min(64, fit / 2 / 16 * 16); }
  else if (fit >= 16) { P->route_bufs = 1; P->route_spans = 16; }
  else if (c.route_dim != 32 && fit >= 8) { P->route_bufs = 1; P->route_spans = fit; }
  else { if (why) *why = "routing-table staging does not fit the team's shared memory"; return false; }
  return true;
}

int fused_warps() { return kFusedWarps; }

template <int G>
static cudaError_t launch_fused_g(const FusedParams& P, size_t smem, int grid, int threads, cudaStream_t s, bool pdl) {
  cudaError_t e = cudaFuncSetAttribute(fused_layer_kernel<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3(grid); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, fused_layer_kernel<G>, P);
}

template <int G>
static cudaError_t occupancy_g(size_t smem, int threads, int* ctas_per_sm) {
  cudaError_t e = cudaFuncSetAttribute(fused_layer_kernel<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, fused_layer_kernel<G>, threads, smem);
}

#define SEKV_DISPATCH_G(G, CALL)                 \
  switch (G) {                                   \
    case 1: e = CALL(1); break;                  \
    case 2: e = CALL(2); break;                  \
    case 3: e = CALL(3); break;                  \
    case 4: e = CALL(4); break;                  \
    case 5: e = CALL(5); break;                  \
    case 6: e = CALL(6); break;                  \
    case 7: e = CALL(7); break;                  \
    case 8: e = CALL(8); break;                  \
    default: e = cudaErrorInvalidValue; break;   \
  }

// The persistent kernel spins on counters published by other CTAs: every CTA of the grid must be resident.
// Returns how many CTAs of the fused kernel one SM can hold with the current device state.
cudaError_t fused_occupancy(const sekv_handle* h, int* ctas_per_sm) {
  const size_t smem = (size_t)kFusedWarps * kRegionBytes;
  cudaError_t e;
#define OCC(GG) occupancy_g<GG>(smem, kFusedThreads, ctas_per_sm)
  SEKV_DISPATCH_G(h->G, OCC)
#undef OCC
  return e;
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
  P.grp = (const int2*)ws(h, h->F.off_bg_part);
  P.partials = (float*)ws(h, h->F.off_partials1);
  P.zdesc = (ZDescG*)ws(h, h->F.off_zdesc) + (size_t)layer * c.max_seqs * c.n_kv_heads * (std::max(c.k_cap, 1) + std::max(c.prefetch, 0));
  P.ctrs = (int32_t*)ws(h, h->F.off_ctrs) + (size_t)layer * h->F.ctrs_per_layer;
  P.ctrs_set = (h->F.ctrs_per_layer - 4) / 2;
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
  // Speculative prefetch (whole-step launches): the candidates of layer l are copied by the kernel of layer
  // l + 1 (those of the last layer by layer 0 of the next step; sekv_api.cu covers the cases without one).
  if (!((mode & FM_ROUTE) && (mode & FM_ATTN))) P.prefetch = 0;
  if ((mode & FM_ROUTE) && (mode & FM_ATTN) && c.n_layers > 1 && c.prefetch > 0 && c.k_cap > 0) {
    // with three layers or more: the layer two launches back, copied before the dependency wait (fused_layer_kernel);
    // layers 0 and 1 carry the last two layers' copies of the previous step
    P.pf_early = c.n_layers >= 3 ? 1 : 0;
    const int pl = (layer + c.n_layers - (P.pf_early ? 2 : 1)) % c.n_layers;
    P.pf_lv = layer_view(h, pl);
    P.pf_plan_counts = (const int32_t*)ws(h, h->F.off_plan_counts) + (size_t)pl * c.max_seqs * c.n_kv_heads * 2;
  }
  P.kc = std::max(c.k_cap, 1) + std::max(c.prefetch, 0);
  P.BG = h->n_seqs * c.n_kv_heads;
  P.Hq = c.n_q_heads; P.Hkv = c.n_kv_heads; P.dp = c.route_dim; P.ways = c.cache_ways;
  P.mask_words = h->mask_words; P.spans_cap = (int)h->lay.spans_cap; P.m_tot = h->m_tot;
  P.out_bf16 = c.out_dtype == SEKV_BF16;
  P.slot_bytes = h->lay.slot_bytes;
  P.ent_head_stride = (size_t)h->lay.rows_cap * kD;
  P.route_head_stride = (size_t)h->lay.spans_cap * c.route_dim;
  if (!fused_geometry(h, &P, nullptr)) return cudaErrorInvalidConfiguration;
  P.zmask2 = (uint2*)ws(h, h->F.off_zmask2) + (size_t)layer * c.max_seqs * c.n_kv_heads * h->mask_words;
  P.zway = (uint2*)ws(h, h->F.off_zway) + (size_t)layer * c.max_seqs * c.n_kv_heads * (std::max(c.k_cap, 1) + std::max(c.prefetch, 0));
  // the chain (a1-a4) runs whenever there is routing to do or a zoom set to plan
  P.has_chain = ((mode & FM_ROUTE) || c.k_cap > 0) ? 1 : 0;
  // layers 1.. of a whole-step launch: the kernel before this one on the stream is the previous layer's of the same
  // step (it writes none of this layer's tables), so the chain's static part, the step stamp and the sequence
  // number may be read before the dependency wait.  Layer 0 follows whatever the caller ran last: no hoisting.
  P.hoist = ((mode & FM_ROUTE) && (mode & FM_ATTN) && layer > 0) ? 1 : 0;
  if ((mode & FM_ROUTE) && (mode & FM_ATTN)) {                  // whole-step launches run the layers in order
    const LayerView nv = layer_view(h, (layer + 1) % c.n_layers);
    P.next_W = (const uint8_t*)nv.W;
    P.next_route = (const uint8_t*)nv.route;
    P.next_W_bytes = (size_t)c.n_q_heads * c.route_dim * kD * 2;
    P.next_route_head_bytes = (size_t)h->m_tot * c.route_dim * 2;
  }
  P.main_end = (mode & FM_ATTN) ? h->n_items : 0;
  const size_t smem = (size_t)kFusedWarps * kRegionBytes;
  const int grid = h->fused_grid, threads = kFusedThreads;
  cudaError_t e;
#define LAUNCH(GG) launch_fused_g<GG>(P, smem, grid, threads, s, h->use_pdl)
  SEKV_DISPATCH_G(h->G, LAUNCH)
#undef LAUNCH
  h->launches += 1;
  return e;
}

cudaError_t launch_prefetch(sekv_handle* h, int layer, cudaStream_t s) {
  const sekv_config& c = h->cfg;
  if (c.prefetch <= 0 || c.k_cap <= 0) return cudaSuccess;
  const size_t smem = std::min<size_t>(round_up_sz((size_t)h->lay.slot_bytes, 128), kBounceBytes);
  dim3 grid(c.prefetch, h->n_seqs * c.n_kv_heads);
  const int32_t* pc = (const int32_t*)ws(h, h->F.off_plan_counts) + (size_t)layer * c.max_seqs * c.n_kv_heads * 2;
  prefetch_kernel<<<grid, 32, smem, s>>>(csr_view(h), layer_view(h, layer), pc, std::max(c.k_cap, 1) + c.prefetch,
                                         c.n_kv_heads, c.cache_ways, (int)h->lay.spans_cap, h->lay.slot_bytes, h->host_dev);
  h->launches += 1;
  return cudaGetLastError();
}

}  // namespace sekv
