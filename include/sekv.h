/*
 * sekv.h -- C ABI of the B200-native SeKV decode hot path (arxiv/paper_2606_31145).
 *
 * The library implements, as hand-written CUDA for sm_100a, the per-decode-step path of SeKV
 * (sec. 3.2-3.3, Fig. 2): coarse routing of the query against per-span summaries with
 * top-k zoom-in selection, fetch of the selected spans' low-rank SVD factors from a pinned-host
 * store into a device factor cache, and one attention pass over the mixed-resolution memory
 * (full-resolution anchors, one coarse entry per unexpanded span, factor-reconstructed tokens of
 * expanded spans) merged by log-sum-exp -- plus the prefill-time construction that feeds it.
 *
 * Conventions
 *  - Plain C, no torch types.  Every pointer says whether it is HOST or DEVICE memory.
 *  - The caller owns all large memory: one device arena and one pinned (page-locked, device-
 *    mapped) host arena handed to sekv_create and borrowed until sekv_destroy.  The library
 *    sub-allocates them with a fixed layout (sekv_get_layout) and allocates nothing large itself.
 *  - Calls are asynchronous on the `main_stream` given in the config unless stated otherwise; the
 *    factor fetch runs on `side_stream`, ordered against the main stream by events.
 *  - Every call returns a sekv_status; nothing throws or aborts across the ABI; on error no output
 *    is written (CUDA launch errors excepted) and sekv_last_error(h) describes the failure.
 *  - One handle must not be used from two threads at once.  There is no CPU fallback: with no
 *    CUDA device every compute call returns SEKV_CUDA.
 *  - Element layouts are row-major with the last index fastest.  `st` = storage dtype of the
 *    config (bf16 or fp32).  Head dimension d_h is 128.
 *
 * Citations are to /root/reference/PAPER.md line numbers (L..), equations and sections.
 */
#ifndef SEKV_H_
#define SEKV_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define SEKV_API __attribute__((visibility("default")))
#else
#define SEKV_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

#define SEKV_VERSION_MAJOR 0
#define SEKV_VERSION_MINOR 1
#define SEKV_HEAD_DIM 128
#define SEKV_MAX_GROUP 8      /* query heads per kv head */
#define SEKV_MAX_RANK 64      /* R_max swept up to 64 in PAPER.md Table 7 */
#define SEKV_MAX_ROUTE_DIM 64
#define SEKV_MAX_SPAN_LEN 1024
#define SEKV_MAX_SPANS_PER_SEQ 8192

typedef enum sekv_status {
  SEKV_OK = 0,
  SEKV_INVALID_ARG = 1,
  SEKV_UNSUPPORTED = 2,
  SEKV_OOM_DEVICE = 3,   /* device arena too small */
  SEKV_OOM_HOST = 4,     /* pinned host arena too small */
  SEKV_CUDA = 5,         /* a CUDA runtime call failed (text in sekv_last_error) */
  SEKV_STATE = 6         /* call out of order, e.g. decode before build */
} sekv_status;

typedef enum sekv_dtype { SEKV_F32 = 0, SEKV_BF16 = 1 } sekv_dtype;

typedef struct sekv_handle sekv_handle;

/* Static configuration.  Hyper-parameter defaults of the paper: alpha = 1.0, l_min = 16, d' = 32,
 * R_max = 32. */
typedef struct sekv_config {
  int32_t n_layers;          /* L */
  int32_t n_q_heads;         /* H   (query heads; routing is per query head, L158-160) */
  int32_t n_kv_heads;        /* H_kv; H % H_kv == 0, H / H_kv <= SEKV_MAX_GROUP */
  int32_t head_dim;          /* d_h, must be 128 */
  int32_t route_dim;         /* d' (Eq. 3-4), multiple of 8, <= SEKV_MAX_ROUTE_DIM */
  int32_t dtype;             /* sekv_dtype: storage of K/V rows, summaries, W, factors, q */
  int32_t out_dtype;         /* sekv_dtype of the attention output */
  float alpha;               /* boundary sensitivity (L55) */
  int32_t l_min;             /* spans shorter than this stay at full resolution (L108) */
  int32_t r_max;             /* rank cap R_max (Eq. 6), <= SEKV_MAX_RANK */
  int32_t window;            /* last `window` tokens are full resolution (Eq. 17) */
  int32_t max_seqs;          /* B capacity */
  int64_t max_tokens_total;  /* capacity of sum_b n_b (segmentation scratch) */
  int32_t max_spans_total;   /* capacity of sum_b m_b */
  int32_t max_full_total;    /* capacity of sum_b A_b (anchors + short runs + window) */
  int32_t max_span_len;      /* <= SEKV_MAX_SPAN_LEN; longer runs make build fail UNSUPPORTED */
  int32_t k_cap;             /* max zoomed spans per (sequence, kv head) and step */
  int32_t cache_ways;        /* device factor-cache slots per (layer, sequence, kv head), >= k_cap + prefetch */
  int32_t prefetch;          /* speculative prefetch depth: the `prefetch` next-best spans by routing score of a
                                layer-step that are not resident are given a slot and copied host -> cache off the
                                critical path: in sekv_decode_step by the layer kernel two launches later (before its
                                dependency wait; one launch later with two layers), else by a copy kernel before the
                                layer's cache is read again */
  int32_t stage1_ctas;       /* generic path: stage-1 grid; 0 = auto (multiple of the SM count) */
  int32_t item_rows;         /* fused path: entry rows per POOL work item, multiple of 16 (COARSE items: min(this, 64)); 0 = one round over the streaming warps */
  int32_t zoom_spans_per_item; /* reserved (the fused path runs one expanded span per ZOOM work item) */
  int32_t use_graph;         /* 1: sekv_decode_step replays a captured CUDA graph */
  int32_t impl;              /* 0 = auto (bf16: the fused layer kernel), 1 = force the generic multi-kernel path */
  void* main_stream;         /* cudaStream_t; NULL = legacy default stream */
  void* side_stream;         /* cudaStream_t for the factor fetch; NULL = created by the library */
} sekv_config;

/* Byte offsets (into the device arena unless named host_) and strides of every table, for tests,
 * export and debugging.  All strides in BYTES.  Filled by sekv_get_layout. */
typedef struct sekv_layout {
  int64_t esize;                 /* bytes per storage element */
  int64_t rows_cap;              /* R_cap = max_full_total + max_spans_total (unified entry rows) */
  int64_t spans_cap;
  /* layer-independent CSR tables */
  int64_t seq_tok_off;           /* int64 [B+1] token offsets */
  int64_t seq_row_off;           /* int32 [B+1] first entry row of each sequence */
  int64_t seq_span_off;          /* int32 [B+1] first span of each sequence */
  int64_t seq_pool_cnt;          /* int32 [B]   A_b */
  int64_t span_len;              /* int32 [m_tot] |S| */
  int64_t span_tok_start;        /* int64 [m_tot] global token index of the span's first token */
  int64_t ln_len;                /* float [m_tot] ln|S| */
  int64_t pool_tok;              /* int64 [A_tot] global token index of each full-resolution token */
  /* per layer */
  int64_t ent_k, ent_v;          /* st [L][H_kv][R_cap][128]: per sequence rows = A_b pool tokens then m_b coarse means */
  int64_t ent_layer_stride, ent_head_stride;
  int64_t route;                 /* st [L][H][spans_cap][d'] routing summaries K_bar */
  int64_t route_layer_stride, route_head_stride;
  int64_t w;                     /* st [L][H][d'][128] */
  int64_t w_layer_stride;
  int64_t dir_off;               /* int64 [L][H_kv][spans_cap] byte offset of the span's blob in the host arena */
  int64_t dir_rank;              /* int32 [L][H_kv][spans_cap] r_K | r_V << 8 | |S| << 16 */
  int64_t dir_layer_stride_elems;
  /* device factor cache */
  int64_t cache_tags;            /* int32 [L][B][H_kv][ways] span id or -1 */
  int64_t cache_stamps;          /* uint32 same shape, step stamp of last use */
  int64_t cache_slots;           /* bytes [L][B][H_kv][ways][slot_bytes] */
  int64_t slot_bytes;
  int64_t host_bytes_used;       /* bytes of the pinned host arena holding factor blobs */
  int64_t device_bytes_total;
} sekv_layout;

/* Counters accumulated since sekv_reset_stats (device-side, read back synchronously). */
typedef struct sekv_stats {
  uint64_t layer_steps;          /* sekv_decode_attn calls (or layers of sekv_decode_step) */
  uint64_t zoomed_spans;         /* (sequence, kv head, span) expansions */
  uint64_t cache_hits;
  uint64_t cache_misses;
  uint64_t h2d_bytes;            /* DEMAND-miss factor bytes read from the pinned host store (Eq. 20) */
  uint64_t factor_bytes_algo;    /* sum over expansions of (r_K+r_V)(|S|+d_h) b + 4(r_K+r_V): Eq. 18 with fp32 sigma */
  uint64_t coarse_rows_skipped;  /* coarse entries replaced by their tokens (= zoomed_spans) */
  uint64_t prefetched_spans;     /* blobs copied by the speculative prefetch (only those that were given a slot) */
  uint64_t kernel_launches;      /* kernels launched or graph nodes replayed by this handle */
  uint64_t prefetch_h2d_bytes;   /* bytes of the blobs copied by the speculative prefetch */
} sekv_stats;

/* Capacities a caller needs BEFORE sekv_create (sekv_build_sizes). */
typedef struct sekv_sizes {
  int64_t tokens_total;          /* sum_b n_b */
  int32_t spans_total;           /* sum_b m_b: exact when H was given, else the bound sum_b floor(n_b / l_min) */
  int32_t full_total;            /* sum_b A_b: exact when H was given, else the bound sum_b n_b */
  int32_t max_spans_per_seq;
  int32_t max_span_len;          /* longest span (exact), else min(SEKV_MAX_SPAN_LEN, longest sequence) */
  int32_t exact;                 /* 1 when computed from H by the segmentation rule */
  int64_t host_bytes;            /* pinned factor store: all layers, kv heads and spans at rank min(r_max, |S|) */
} sekv_sizes;

/* Prefactored build input: the caller supplies the factors instead of dense K/V (skips Eq. 6's
 * SVD; needed to stage 128K x 32 layers where dense K/V would be 68.7 GB).  All DEVICE pointers.
 * The span rows of K (V) are DEFINED as tokU diag(S) Vt.  Token and span axes are the
 * concatenation of the batch's sequences / spans in order; the span axis must agree with what the
 * segmentation rule finds in H (else SEKV_STATE). */
typedef struct sekv_factors {
  int32_t rank_in;             /* r: column count of tokU*, S*, row count of Vt* */
  const void* tokUK;           /* st [H_kv][sum_n][r]  row t = left-factor row of token t (pool rows ignored) */
  const float* SK;             /* f32 [H_kv][m_tot][r] */
  const void* VtK;             /* st [H_kv][m_tot][r][128] */
  const void* tokUV;
  const float* SV;
  const void* VtV;
  const int32_t* rank_k;       /* int32 [H_kv][m_tot] retained rank per span (<= r); NULL = min(r, |S|) */
  const int32_t* rank_v;
  const void* Kfull;           /* st [H_kv][A_tot][128] full-resolution tokens in position order */
  const void* Vfull;
  int32_t a_tot;               /* A_tot the caller laid Kfull/Vfull out for (checked) */
  int32_t m_tot;               /* m_tot the caller laid S/Vt out for (checked) */
} sekv_factors;

/* ---- lifecycle --------------------------------------------------------------------------- */
SEKV_API const char* sekv_version(void);
SEKV_API const char* sekv_status_string(sekv_status s);

/* Bytes of device arena needed for `cfg`; also the factor-cache slot size.  HOST pointers. */
SEKV_API sekv_status sekv_device_arena_bytes(const sekv_config* cfg, size_t* device_bytes, size_t* slot_bytes);

/* Bytes one span's factor blob occupies in the host arena / a cache slot (padded layout, see
 * DESIGN.md section 6): ranks padded to 8, |S| padded to 16.  Pure function. */
SEKV_API size_t sekv_blob_bytes(int32_t dtype, int32_t span_len, int32_t rank_k, int32_t rank_v);

/* Sizes for a batch before any handle exists.  cfg: the static fields (n_layers, heads, dtype, alpha, l_min,
 * r_max, window; capacities are ignored).  seq_tok_off: HOST int64 [n_seqs+1].  H: DEVICE f32 [sum_n] surprisal, or
 * NULL.  With H the segmentation rule of sekv_build_spans (L55, L108, Eq. 17) is run on the GPU (temporary
 * cudaMalloc scratch of ~6 bytes per token, synchronous) and the counts are exact; without it they are upper
 * bounds from the token counts alone (m_b <= n_b / l_min, A_b <= n_b).  spans_per_seq / pool_per_seq: HOST int32
 * [n_seqs] outputs (nullable; bounds when H is NULL).  The caller copies spans_total / full_total /
 * max_span_len (rounded up as it likes) into sekv_config and sizes the pinned host arena with host_bytes. */
SEKV_API sekv_status sekv_build_sizes(const sekv_config* cfg, int32_t n_seqs, const int64_t* seq_tok_off, const float* H,
                             sekv_sizes* out, int32_t* spans_per_seq, int32_t* pool_per_seq);

/* device_arena: DEVICE, 256-byte aligned, >= sekv_device_arena_bytes.  host_arena: HOST, pinned and
 * device-mapped (cudaHostAlloc / torch pin_memory), holds the SVD factor store (PAPER.md L106,
 * L110 "low-rank SVD bases ... reside on CPU").  Zeroes the control tables (synchronous). */
SEKV_API sekv_status sekv_create(const sekv_config* cfg, void* device_arena, size_t device_bytes,
                        void* host_arena, size_t host_bytes, sekv_handle** out);
SEKV_API void sekv_destroy(sekv_handle* h);
SEKV_API const char* sekv_last_error(const sekv_handle* h);

/* ---- a0: prefill-time construction (sec. 3.1-3.2) ---------------------------------- *
 * sekv_build_spans: for one layer and the whole batch,
 *   - (first call only) segmentation from surprisal: boundary iff H_t > mu + alpha*sigma, boundary
 *     tokens are anchors, runs between anchors are spans, runs < l_min and the last `window`
 *     tokens stay full resolution (L55, L108, Eq. 17); fills the CSR tables;
 *   - gathers full-resolution K/V rows (L55, L110);
 *   - surprisal weights w_t (Eq. 2), coarse means k_bar, v_bar (L81), routing summaries
 *     K_bar = normalize(sum w_t W K_t) per query head (Eq. 3);
 *   - truncated SVD of each span's K and V, R = min(|S|, d_h, rank_cap) (Eq. 6, Eq. 8 with binary
 *     gates), written as factor blobs into the pinned host arena (L106).
 * seq_tok_off: HOST int64 [n_seqs+1].  H: DEVICE f32 [sum_n] (may be NULL after the first layer).
 * K, V: DEVICE st [H_kv][sum_n][128].  W: DEVICE st [H][d'][128] for this layer.
 * rank_cap <= cfg.r_max (0 = cfg.r_max).  spans_per_seq / pool_per_seq: HOST int32 [n_seqs]
 * outputs (nullable).  Synchronises the main stream.  Layers may be built in any order; all layers
 * must be built before decoding. */
SEKV_API sekv_status sekv_build_spans(sekv_handle* h, int32_t layer, int32_t n_seqs, const int64_t* seq_tok_off,
                             const float* H, const void* K, const void* V, const void* W,
                             int32_t rank_cap, int32_t* spans_per_seq, int32_t* pool_per_seq);

/* Same, with caller-supplied factors (no SVD). */
SEKV_API sekv_status sekv_build_spans_prefactored(sekv_handle* h, int32_t layer, int32_t n_seqs,
                                         const int64_t* seq_tok_off, const float* H,
                                         const sekv_factors* f, const void* W,
                                         int32_t* spans_per_seq, int32_t* pool_per_seq);

/* Forget all sequences (tables, factor store, cache). */
SEKV_API sekv_status sekv_reset(sekv_handle* h);

/* ---- a1-a3: routing (Eq. 4, 5, 9; budget cap L123) --------------------------------- *
 * q: DEVICE st [B][H][128].  tau: DEVICE f32 [H] thresholds in probability space or NULL (pure
 * top-k).  k: zoom cap per (sequence, kv head); k < 0 = every eligible span (needs k_cap >= m_b).
 * Outputs (DEVICE): logits x [H][m_tot] f32 (the sigmoid's argument, nullable), alpha_tilde
 * [H][m_tot] f32 (nullable), ids int32 [B][H_kv][k_cap] in decreasing-score order (ties to the
 * lower span id; unused entries -1; ids are span indices LOCAL to the sequence), count int32
 * [B][H_kv].  Selection is per kv head on X = max over the group's query heads. */
SEKV_API sekv_status sekv_route(sekv_handle* h, int32_t layer, const void* q, const float* tau, int32_t k,
                       float* logits, float* alpha_tilde, int32_t* ids, int32_t* count);

/* ---- a4-a7: factor fetch + mixed-resolution attention (Fig. 2, Eq. 8) ---- *
 * q: DEVICE st [B][H][128].  ids/count: DEVICE, as written by sekv_route or any caller-chosen zoom
 * set (local span ids, no duplicates, count <= k_cap).  out: DEVICE out_dtype [B][H][128].
 * lse: DEVICE f32 [B][H] natural-log-sum-exp of each head's softmax (nullable).
 * Steps: residency lookup in the device factor cache and slot assignment (LRU per (layer,
 * sequence, kv head)); copy of missing blobs pinned-host -> slot on the side stream; stage 1:
 * online-softmax partials over pool tokens and unexpanded coarse entries (+ln|S|); stage 2: partials
 * over the expanded spans' tokens through the factored form logits = (U Sigma)(V^T q); log-sum-exp
 * combine. */
SEKV_API sekv_status sekv_decode_attn(sekv_handle* h, int32_t layer, const void* q, const int32_t* ids,
                             const int32_t* count, void* out, float* lse);

/* One decode step over all layers: for l in 0..L-1 { route; decode_attn }.  q: DEVICE st
 * [L][B][H][128]; tau: DEVICE f32 [L][H] or NULL; out: DEVICE out_dtype [L][B][H][128]; lse: DEVICE
 * f32 [L][B][H] or NULL.  With cfg.use_graph the launch sequence is captured once per distinct
 * argument tuple and replayed. */
SEKV_API sekv_status sekv_decode_step(sekv_handle* h, const void* q, const float* tau, int32_t k, void* out,
                             float* lse);

/* Zoom sets chosen by the last sekv_decode_step for `layer`: copies ids [B][H_kv][k_cap] and count
 * [B][H_kv] (DEVICE int32 outputs, same format as sekv_route) on the main stream. */
SEKV_API sekv_status sekv_last_zoom_ids(sekv_handle* h, int32_t layer, int32_t* ids, int32_t* count);

/* Same through HOST buffers (pinned recommended): copies q host->device, runs the step, copies
 * out (and lse if not NULL) device->host, and waits for completion.  tau stays a DEVICE pointer. */
SEKV_API sekv_status sekv_decode_step_host(sekv_handle* h, const void* q_host, const float* tau, int32_t k,
                                  void* out_host, float* lse_host);

/* ---- introspection ------------------------------------------------------------------------- */
SEKV_API sekv_status sekv_get_layout(const sekv_handle* h, sekv_layout* out);       /* HOST out */
SEKV_API sekv_status sekv_get_stats(sekv_handle* h, sekv_stats* out);               /* HOST out; synchronises */
SEKV_API sekv_status sekv_reset_stats(sekv_handle* h);
SEKV_API sekv_status sekv_cache_flush(sekv_handle* h);                              /* drop all cached factors */
/* Algorithmic HBM bytes of one layer-step excluding the zoomed factors: routing
 * summaries + 4m, pool rows, q and out, W; coarse rows are counted in full (the per-step
 * correction for skipped coarse rows and the factor bytes come from sekv_stats). HOST out. */
SEKV_API sekv_status sekv_static_bytes_per_layer(const sekv_handle* h, uint64_t* bytes);
/* Per-kernel timing with CUDA events recorded on the launching stream around every kernel of
 * sekv_route / sekv_decode_attn / sekv_decode_step (non-graph launches only; a graph replay is not
 * instrumented).  Classes: 0 route (a1-a3), 1 plan (a4 residency), 2 fetch (a4 copy, side stream),
 * 3 stage 1 (a5), 4 stage 2 (a6), 5 combine (a7) -- the generic multi-kernel path -- and 6 the fused
 * layer kernel (a1-a7 in one launch, bf16 path), 7 the stand-alone prefetch copy kernel.
 * sekv_get_kernel_times synchronises, writes the summed milliseconds and launch counts per class since
 * the last call (HOST arrays of SEKV_N_KERNEL_CLASSES) and clears. */
#define SEKV_N_KERNEL_CLASSES 8
SEKV_API sekv_status sekv_set_profiling(sekv_handle* h, int32_t on);
SEKV_API sekv_status sekv_get_kernel_times(sekv_handle* h, double* ms, uint64_t* launches);
/* Work-item trace of the fused layer kernel (a debugging and tuning instrument; off by default).
 * `buf` is a DEVICE buffer of capacity_items records of 64 bytes, borrowed until the next call
 * (buf = NULL switches tracing off).  Every launch of layer l overwrites record l * (*n_items + groups) + i
 * (groups = sequences x kv heads; the team's selection / plan of group g is item *n_items + g) for work item i with
 * { int32 kind, int32 group, uint16 sm, uint16 warp, int32 0, uint64 t_begin_ns, uint64 t_end_ns,
 *   uint64 mark_ns[4] } (%globaltimer; mark 0 = end of the item's dependency wait);
 * items past the capacity are not recorded.  HOST out *n_items: items per full layer launch. */
SEKV_API sekv_status sekv_set_trace(sekv_handle* h, void* buf, int64_t capacity_items, int32_t* n_items);
/* Number of stage-1 work chunks (CTAs) and partial slots per query head; HOST outs. */
SEKV_API sekv_status sekv_get_schedule(const sekv_handle* h, int32_t* stage1_ctas, int32_t* parts_per_head);
/* Number of CUDA graphs sekv_decode_step holds (one per distinct argument tuple; a replay adds none).  HOST out. */
SEKV_API sekv_status sekv_graph_count(const sekv_handle* h, int32_t* count);
/* Which kernels the built batch runs on.  *fused = 1: the persistent fused layer kernel (bf16 path, one launch
 * per layer-step); 0: the generic multi-kernel path, and *reason (a string owned by the handle, valid until the
 * next build / reset) says why -- fp32 storage, impl = 1, a sequence with too many spans for the team's shared
 * memory, tables too small, the kernel not resident on this device.  Nothing switches paths silently: callers
 * that depend on the fused kernel's speed check this after the first sekv_build_spans call.  HOST outs. */
SEKV_API sekv_status sekv_get_path(const sekv_handle* h, int32_t* fused, const char** reason);
/* Decode one span's factor blob from the pinned host store into plain row-major fp32 HOST arrays (format
 * decoding only; the blob layout -- mma fragment order, DESIGN.md section 5 -- lives in one place, the
 * library).  span is LOCAL to sequence seq.  Outputs (nullable): UK [|S|][r_K], sK [r_K], VtK [r_K][128],
 * UV [|S|][r_V], sV [r_V], VtV [r_V][128]; *len, *rank_k, *rank_v always.  Call with NULL arrays first to
 * learn the shapes.  *pad_zero = 1 iff every padding element of the blob is zero. */
SEKV_API sekv_status sekv_export_span_factors(sekv_handle* h, int32_t layer, int32_t seq, int32_t kv_head, int32_t span,
                                     int32_t* len, int32_t* rank_k, int32_t* rank_v, float* UK, float* sK,
                                     float* VtK, float* UV, float* sV, float* VtV, int32_t* pad_zero);

/* The segmentation counts of sekv_build_sizes (rule of L55, L108, Eq. 17 window) for callers that may not call
 * cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid allocation.  This entry
 * point allocates NOTHING (no cudaMalloc / cudaFree / allocating library routine, no host allocation): the ~6
 * bytes per token of scratch that sekv_build_sizes takes from a temporary cudaMalloc live in a file-scope
 * `static __device__` array of the library, sized for SEKV_STATIC_MAX_TOKENS tokens in SEKV_STATIC_MAX_SEQS
 * sequences (6.02 MiB; every GPU that loads the library holds it until the process exits).
 *   cfg: alpha, l_min, window are read (the static fields of sekv_build_sizes; capacities ignored).
 *   seq_tok_off: HOST int64 [n_seqs+1], seq_tok_off[0] = 0, increasing (copied to the scratch on `stream`).
 *   H: DEVICE f32 [seq_tok_off[n_seqs]] surprisal.
 *   counts: DEVICE int32 [n_seqs][2] output = (full-resolution pool tokens A_b, spans m_b) per sequence.
 *   too_long: DEVICE int32 [1] output = 1 iff some run exceeds SEKV_MAX_SPAN_LEN (sekv_build_sizes returns
 *   UNSUPPORTED there), else 0.
 *   stream: cudaStream_t of the CURRENT device (0 = default stream).  Asynchronous: outputs are ready when the
 *   stream reaches the end of this call's work.
 * Errors: INVALID_ARG (NULL pointer, bad cfg / offsets) and UNSUPPORTED ("... exceeds SEKV_STATIC_MAX_...", nothing
 * launched, outputs untouched) -- the message is returned by sekv_static_last_error().  CUDA for launch failures.
 * Every call on a device shares that device's array, which keeps the previous call's contents (this call needs
 * nothing pre-zeroed beyond what it clears itself): calls that overlap on the GPU -- two streams, or two threads --
 * RACE; serialise them (same stream, or an event between them). */
#define SEKV_STATIC_MAX_TOKENS (1 << 20)
#define SEKV_STATIC_MAX_SEQS 1024
SEKV_API sekv_status sekv_segment_counts_static(const sekv_config* cfg, int32_t n_seqs, const int64_t* seq_tok_off,
                                                const float* H, int32_t* counts, int32_t* too_long, void* stream);
/* Message of the calling thread's last failed sekv_segment_counts_static call ("" if none). */
SEKV_API const char* sekv_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SEKV_H_ */
