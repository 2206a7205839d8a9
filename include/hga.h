/*
 * hga.h -- C ABI of the B200-native (sm_100a) Hierarchical Global Attention prefill hot path.
 *
 * Method: arxiv/paper_2606_30709 ("Hierarchical Global Attention", PAPER.md).  The library exports the four
 * stages BASELINE.json's north_star names, as calls over device-resident tensors:
 *
 *   hga_rope             S0  RoPE on Q + chunk-shared pooled query            PAPER.md:62; 33, 45, 97
 *   hga_build_summaries  S1  RoPE on K + mixed-RoPE chunk / group summaries   PAPER.md:80-89 (section 3.2)
 *   hga_route            S2  chunk top-K_c over the middle context            PAPER.md:95-97 (section 3.3)
 *                        S3  group refinement, top-K_g inside those chunks
 *   hga_attend           S4  exact softmax attention over sink U local U routed U current tokens (GQA)
 *                                                                             PAPER.md:103-109 (section 3.4), Eq. (1)
 *   hga_prefill          S0..S4 enqueued back to back on one stream
 *   hga_host_*           the same path for HOST buffers (H2D, S0..S4, D2H), used for end-to-end timing
 *
 * Conventions (all entry points):
 *   - Tensor pointers are DEVICE pointers owned by the caller unless the argument name ends in `_host`.
 *     Tensors are contiguous, head_dim fastest, and 16-byte aligned.  The library never allocates, frees or
 *     synchronises in the device-pointer calls; work is enqueued on `stream` (a cudaStream_t passed as void*,
 *     NULL = the legacy default stream).  Scratch memory comes from the caller (hga_workspace_bytes).
 *   - Layouts ("[...]" lists dims slowest to fastest):
 *       Q       [batch, n_q_heads,  seq, head_dim]   io_dtype
 *       K, V    [batch, n_kv_heads, seq, head_dim]   io_dtype
 *       pooled  [batch, n_kv_heads, seq/chunk, head_dim]            float
 *       chunk_sum  [batch, n_kv_heads, seq/chunk, head_dim]         float
 *       group_sum  [batch, n_kv_heads, seq/group, head_dim]         float
 *       chunk_idx / chunk_score  [batch, n_kv_heads, seq/chunk, topk_chunks]   int32 / float
 *       group_idx / group_score  [batch, n_kv_heads, seq/chunk, topk_groups]   int32 / float
 *       n_chunks / n_groups      [batch, n_kv_heads, seq/chunk]                int32
 *       out     [batch, n_q_heads, seq, head_dim]    out_dtype;   lse [batch, n_q_heads, seq] float
 *     Index lists are ascending, -1 padded after the first n_* entries.  Query head h uses KV head
 *     h / (n_q_heads / n_kv_heads) (GQA).
 *   - Errors are return codes; nothing throws and there is no global state.  Shape, divisibility, null and
 *     alignment problems are rejected on the host before any launch (HGA_ERR_INVALID_ARG / _UNSUPPORTED /
 *     _WORKSPACE); a failed launch maps to HGA_ERR_CUDA.  There is no CPU fallback: without a CUDA device every
 *     compute call returns HGA_ERR_CUDA.
 *   - Non-finite inputs are undefined behaviour (the CPU oracle rejects them).
 */
#ifndef HGA_H_
#define HGA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define HGA_API __attribute__((visibility("default")))
#else
#define HGA_API
#endif

typedef enum {
  HGA_OK = 0,
  HGA_ERR_INVALID_ARG = 1, /* null pointer, bad shape, misaligned pointer */
  HGA_ERR_UNSUPPORTED = 2, /* valid request outside what the kernels implement (e.g. head_dim not in {64,128}) */
  HGA_ERR_WORKSPACE = 3,   /* workspace missing or too small */
  HGA_ERR_CUDA = 4         /* CUDA runtime / launch failure, or no device */
} hga_status;

typedef enum { HGA_F32 = 0, HGA_BF16 = 1 } hga_dtype;

/* How a query block scores a routing candidate (see hga_params). */
typedef enum { HGA_ROUTE_MEAN = 0, HGA_ROUTE_MAX = 1, HGA_ROUTE_MAX_FP64 = 2 } hga_route_mode;

/* hga_params.flags */
typedef enum {
  /* N2: hga_prefill / hga_prefill_window / hga_host_prefill need not materialise the rotated
   * queries.  S0 then only pools them (q_rot is not written and may be NULL), and S4 reads q_raw and applies RoPE
   * to every query tile in shared memory, with the same fp32 arithmetic and the same single rounding to
   * bf16 -- so 2 * |Q| bytes of HBM traffic (the Q_rot write and its read) disappear.  Conditions: io_dtype bf16, whole
   * 64-token blocks, route_mode HGA_ROUTE_MEAN (the max rule reads q_rot), attend_impl HGA_ATTEND_AUTO or
   * HGA_ATTEND_TCGEN05; anything else returns HGA_ERR_UNSUPPORTED (call again without the flag).  The (cos, sin) of a
   * position is formed as the product of two table entries (block start x offset in the block), 2-3 ulp(fp32) instead of
   * 1: a rotated query can differ from S0's by one bf16 rounding step in rare cases. */
  HGA_FLAG_FUSE_Q_ROPE = 1
} hga_flag;

/* Which S4 kernel hga_attend launches. */
typedef enum {
  HGA_ATTEND_AUTO = 0,    /* bf16 -> tcgen05/TMEM kernel (HGA_ATTEND_TCGEN05), f32 -> SIMT fp32 kernel */
  HGA_ATTEND_SIMT = 1,    /* fp32 FMA kernel (any io_dtype): the 1e-4 path for fp32 inputs, and a cross-check */
  HGA_ATTEND_TCGEN05 = 2, /* TMA gather + tcgen05.mma with TMEM accumulators (bf16 inputs only): the persistent
                             kernel; falls back to HGA_ATTEND_TCGEN05_ITEM when the key list does not fit in
                             shared memory beside the tiles */
  HGA_ATTEND_TCGEN05_ITEM = 3, /* the same arithmetic, one (unit, tile pair) per CTA, no cross-item pipelining */
  HGA_ATTEND_TCGEN05_PAIR = 4  /* one CTA pair (2-CTA cluster, tcgen05.mma.cta_group::2) per (batch, kv head, block)
                                  unit: bf16, head_dim 128, groups of exactly 8 query heads; HGA_ERR_UNSUPPORTED
                                  otherwise.  Same results bit for bit as HGA_ATTEND_TCGEN05; measured slower, so
                                  HGA_ATTEND_AUTO does not pick it */
} hga_attend_impl;

/*
 * Problem description (section 3; notation of SURVEY.md section 8).
 *   chunk C must be 64; group g_s must divide chunk and be a multiple of 16 (16 in the paper).
 *   seq must be a multiple of chunk: only closed chunks are summarised.
 *   n_sink F / n_local L: always-visible first / recent chunks.  The immediately preceding chunk is
 *   force-included, i.e. L_eff = max(L, 1).
 *   topk_chunks K_c / topk_groups K_g: route budgets.  K_g = K_c * chunk/group reproduces the
 *   "Qwen3 exact-token variant" (whole chunks opened).  Fewer candidates than budget -> all are taken.
 *   n_hi_chunk / n_hi_group: number of leading (highest-frequency) RoPE pairs that use "rotate per token, then
 *   average"; the remaining pairs use "average raw keys, then rotate at the span's middle position"
 *   (PAPER.md:84-87).  -1 selects the default: pairs whose wavelength 2*pi/theta_i is <= the span length.
 *   RoPE: pair i = (x[i], x[i + head_dim/2]), theta_i = rope_base^(-2i/head_dim), position of token t = pos0 + t.
 *   softmax_scale 0 -> 1/sqrt(head_dim) (Eq. 1).
 *   rope_pos_mod (variant of PAPER.md:259-264, "p <- p mod 65536"): when > 0, every position that enters a rotation
 *   (Q, K, both summary rules) is wrapped modulo it; the routing algorithm is unchanged.  It and pos0 must then be
 *   multiples of `chunk`, so that no chunk or group straddles a wrap (its middle position is the wrapped start +
 *   (S-1)/2); otherwise HGA_ERR_INVALID_ARG.  0 = off.
 *   route_mode (variant; PAPER.md:33, 45, 97 do not say how a block's 64*G queries become one routing score):
 *   HGA_ROUTE_MEAN = dot product with the pooled query (= mean of the per-query scores), the default;
 *   HGA_ROUTE_MAX = the maximum over the block's per-query scores, each the dot product of a rotated query AS STORED
 *   (rounded to io_dtype) with the summary, in fp64 (d ascending, one fma chain).  hga_prefill honours it; the
 *   stand-alone call is hga_route_max.  Whole query blocks only.
 *   HGA_ROUTE_MAX_FP64 = the same rule with every (query, candidate) pair scored on the fp64 pipe: a (64*G) x candidates
 *   x head_dim contraction per block (c5: 29 ms).  HGA_ROUTE_MAX returns the same lists and scores bit for bit, faster
 *   (c5: 1.7 ms): for bf16 I/O, head_dim 64/128, G <= 8, K_c <= 64 and more than 128 blocks, a bf16 hi/lo tcgen05
 *   contraction scores every pair approximately with a proven error bound, and only the candidates that can still reach
 *   the top-K_c -- and, for each of them, only the query rows that can still hold the maximum -- are re-scored in fp64
 *   (a unit whose near-ties exceed the 128-entry candidate list falls back to the fp64 contraction).  Other shapes run
 *   the fp64 contraction under either value.
 */
typedef struct hga_params {
  int32_t batch, seq, n_q_heads, n_kv_heads, head_dim;
  int32_t chunk, group;
  int32_t n_sink, n_local;
  int32_t topk_chunks, topk_groups;
  int32_t n_hi_chunk, n_hi_group;
  int32_t io_dtype;    /* hga_dtype of Q, K, V (raw and rotated) */
  int32_t out_dtype;   /* hga_dtype of `out` */
  int32_t attend_impl; /* hga_attend_impl */
  int64_t pos0;
  double rope_base;
  float softmax_scale;
  int32_t rope_pos_mod; /* 0 = off */
  int32_t route_mode;   /* hga_route_mode */
  int32_t flags;        /* bit mask of hga_flag values; other bits must be 0 */
} hga_params;

HGA_API const char* hga_status_string(hga_status s);

/* Library version (major*10000 + minor*100 + patch). */
HGA_API int32_t hga_version(void);

/* Default high-frequency pair count for a span of `span` tokens (rule above).  Host arithmetic only. */
HGA_API int32_t hga_default_n_hi(int32_t head_dim, double rope_base, int32_t span);

/* Alternative thresholds for "high-frequency" (the paper gives none): the count of leading pairs for
 * a span of `span` tokens under rule 0 (wavelength 2*pi/theta_i <= span, the default), 1 (the span sweeps at least
 * half a turn: theta_i*span >= pi) or 2 (at least one radian: theta_i*span >= 1).  Pass the result as n_hi_chunk /
 * n_hi_group.  Returns -1 for an unknown rule.  Host arithmetic only. */
HGA_API int32_t hga_n_hi_rule(int32_t head_dim, double rope_base, int32_t span, int32_t rule);

/* Validate `p` without touching the GPU. */
HGA_API hga_status hga_validate(const hga_params* p);

/* Bytes of device scratch hga_route / hga_prefill need for `p`: chunk scores [batch, n_kv_heads, R, seq/chunk] float with
 * R = min(seq/chunk, 1024) -- the route stage runs in slabs of at most 1024 query blocks, so the scratch grows linearly
 * with the sequence past 64K tokens (more under HGA_ROUTE_MAX and HGA_FLAG_FUSE_Q_ROPE, which add their own tables).
 * Host arithmetic only. */
HGA_API hga_status hga_workspace_bytes(const hga_params* p, size_t* bytes);

/*
 * S0.  x_rot[b,h,t,:] = RoPE(x_raw[b,h,t,:], pos0 + t) for a [batch, n_heads, seq, head_dim] tensor,
 * computed in fp32 with fp64 range reduction of the angle and rounded once to io_dtype.  x_rot may alias x_raw.
 * If `pooled` is non-null (then n_heads must be a multiple of n_kv_heads): pooled[b,kv,j,:] = mean over the
 * chunk's tokens and the n_heads/n_kv_heads heads of KV group kv of the UN-ROUNDED rotated vectors -- the one
 * routing query of block j (chunk-shared routing; per KV head).
 */
HGA_API hga_status hga_rope(const hga_params* p, const void* x_raw, int32_t n_heads, void* x_rot, float* pooled,
                            void* stream);

/*
 * S1.  k_rot = RoPE(k_raw) (rounded once to io_dtype; may alias k_raw; may be NULL to skip the
 * store), and for every chunk / group span the mixed-RoPE summary (mean; middle position = start + (S-1)/2),
 * accumulated in fp64 from un-rounded fp32 values and stored as float.  chunk_sum / group_sum may be NULL.
 */
HGA_API hga_status hga_build_summaries(const hga_params* p, const void* k_raw, void* k_rot, float* chunk_sum,
                                       float* group_sum, void* stream);

/*
 * S2 + S3.  For every (b, kv, block j): candidates are the middle chunks
 * c in [n_sink, j - max(n_local,1)); score(c) = <q_pooled[b,kv,j], chunk_sum[b,kv,c]> (fp64 accumulation of fp32
 * inputs, stored as float); the min(K_c, #candidates) highest are kept (ties -> lower index).  Then the
 * chunk/group groups of every kept chunk are scored against group_sum the same way and the min(K_g, #) highest
 * kept.  Outputs as listed at the top; chunk_score / group_score / n_chunks / n_groups may be NULL.
 * If topk_groups == 0 the group stage is skipped (group_idx may be NULL).
 * workspace: at least hga_workspace_bytes(p) bytes, 16-byte aligned.
 */
HGA_API hga_status hga_route(const hga_params* p, const float* q_pooled, const float* chunk_sum,
                             const float* group_sum, int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks,
                             int32_t* group_idx, float* group_score, int32_t* n_groups, void* workspace,
                             size_t workspace_bytes, void* stream);

/*
 * hga_route without a workspace argument and without any allocation, for callers that cannot call cudaMalloc (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid it): the chunk-score matrix lives in a static device
 * array of HGA_ROUTE_STATIC_MAX_BYTES inside the library (every GPU that loads the library holds it until the process
 * exits).  Same arguments, outputs and results as hga_route, bit for bit.  Limit: batch * n_kv_heads * min(seq/chunk, 1024) * (seq/chunk) * 4
 * bytes <= HGA_ROUTE_STATIC_MAX_BYTES (BASELINE.json configs[4], 64K tokens x 4 KV heads, fits exactly); a larger problem
 * returns HGA_ERR_WORKSPACE and launches nothing -- use hga_route with a caller-owned workspace.  HGA_ROUTE_MEAN only.
 * The first call on a device looks the array's address up (cudaGetSymbolAddress, which may load the module: make one
 * call before starting a graph capture).  All calls share the array: calls that overlap on the GPU (different streams,
 * concurrently replayed graphs) race; calls ordered on one stream do not.  Nothing in it has to be cleared between calls.
 */
#define HGA_ROUTE_STATIC_MAX_BYTES (16u << 20)
HGA_API hga_status hga_route_static(const hga_params* p, const float* q_pooled, const float* chunk_sum,
                                    const float* group_sum, int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks,
                                    int32_t* group_idx, float* group_score, int32_t* n_groups, void* stream);

/*
 * S2 + S3 under HGA_ROUTE_MAX / HGA_ROUTE_MAX_FP64 (p->route_mode must be one of them): the same candidate sets, budgets, tie rule and
 * outputs as hga_route, with score(candidate) = max over the 64*G rotated queries of block j (all heads of the GQA
 * group, read from q_rot [B,H_q,N,D] in io_dtype) of <q, summary> in fp64.  hga_route itself rejects HGA_ROUTE_MAX
 * (HGA_ERR_INVALID_ARG): it is given no per-query tensor.  workspace: hga_workspace_bytes(p) bytes (larger in this mode).
 */
HGA_API hga_status hga_route_max(const hga_params* p, const void* q_rot, const float* chunk_sum,
                                 const float* group_sum, int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks,
                                 int32_t* group_idx, float* group_score, int32_t* n_groups, void* workspace,
                                 size_t workspace_bytes, void* stream);

/*
 * S4.  For query row (b,h,t) in block j = t / chunk with kv = h / (n_q_heads/n_kv_heads):
 *   keys = tokens of chunks {0..min(F,j)-1} U {max(0,j-max(L,1))..j-1} U groups group_idx[b,kv,j,:] U {u in chunk j, u <= t}
 *   out  = sum_u softmax_u(softmax_scale * <q_rot, k_rot_u>) v_u      (fp32 accumulation, online softmax)
 *   lse  = log sum_u exp(softmax_scale * <q_rot, k_rot_u>)            (optional, may be NULL)
 * group_idx entries must be -1 or groups of chunks closed before block j; entries inside the sink / local
 * windows are allowed (set union), entries reaching chunk j or later are ignored, duplicate entries are undefined.
 * The list need not be sorted.  Any list is accepted (not only hga_route's), e.g. all earlier groups == dense
 * causal attention.  group_idx may be NULL when topk_groups == 0.
 */
HGA_API hga_status hga_attend(const hga_params* p, const void* q_rot, const void* k_rot, const void* v,
                              const int32_t* group_idx, void* out, float* lse, void* stream);

/*
 * Device buffers of one prefill pass.  q_rot / k_rot may alias q_raw / k_raw (in-place RoPE).  chunk_score,
 * group_score, n_chunks, n_groups and lse may be NULL.
 */
typedef struct hga_buffers {
  const void* q_raw;
  const void* k_raw;
  const void* v;
  void* q_rot;
  void* k_rot;
  float* q_pooled;
  float* chunk_sum;
  float* group_sum;
  int32_t* chunk_idx;
  float* chunk_score;
  int32_t* n_chunks;
  int32_t* group_idx;
  float* group_score;
  int32_t* n_groups;
  void* out;
  float* lse;
  void* workspace;
  size_t workspace_bytes;
} hga_buffers;

/* S0..S4 enqueued on `stream`: hga_rope(Q) -> hga_build_summaries(K) -> hga_route -> hga_attend. */
HGA_API hga_status hga_prefill(const hga_params* p, const hga_buffers* buf, void* stream);

/*
 * Streaming step: chunk-by-chunk prefill, single-token decode, ragged prompt tail.
 * The store/router cycle of PAPER.md:158 ("appending a newly closed chunk, reading chunk summaries for routing,
 * fetching group summaries for the second routing level, and gathering exact token K/V") for the token window
 * [t_begin, t_end) of a cache whose capacity is p->seq tokens; "vectorized prefill and chunk-by-chunk decode must
 * agree up to floating-point noise" (Table 7 :291-292).  hga_prefill is the window [0, p->seq).
 *
 * All tensors of `buf` keep the full-capacity layouts above and persist between calls (they ARE the cache).  On
 * entry q_raw / k_raw / v hold the window's rows (k_raw also the earlier rows of a chunk that the window closes);
 * K_rot, V and the summary tables hold what earlier calls left for tokens < t_begin.  The call
 *   - rotates and stores Q_rot / K_rot rows of the window only (S0, S1);
 *   - writes the chunk and group summaries of every chunk the window CLOSES, (c+1)*chunk <= t_end, from the raw keys of
 *     the whole chunk -- an open chunk has no summary;
 *   - routes every query block that intersects the window with q_pooled = mean of the rotated queries of the block's
 *     rows INSIDE the window over the GQA group (reading R17: a whole block gives hga_prefill's pooled query, a single
 *     decode token routes with its own pooled query) against the closed chunks before it (S2, S3); results go to row
 *     j = t / chunk of q_pooled / chunk_idx / group_idx / ... (overwriting what an earlier step of the same block left);
 *   - attends (S4): writes the out / lse rows of the window and no others.  Whole 64-row blocks go to the kernel
 *     hga_attend would pick; a partial block (a window that starts or ends inside a chunk) goes to the fp32 kernels --
 *     steps of up to 4 query rows (decode, short appends) to attend_rows_kernel (key list split over 8 warps, online
 *     softmax per warp, partial results merged), longer partial blocks to the row-masked SIMT tile kernel.
 *     A window that starts inside a chunk must stay inside that chunk (one step of the active chunk).
 * In-place RoPE: q_rot may alias q_raw for any window.  k_rot may alias k_raw ONLY for chunk-aligned windows
 * (t_begin and t_end multiples of chunk): a step that closes a chunk summarises the whole chunk from k_raw, and with
 * the alias earlier partial steps would already have replaced its first rows by rotated keys.
 * Values at positions >= t_end never influence a result and nothing there is written: the future part of the cache
 * may be uninitialised (even NaN).  A chunk is summarised only by the call whose window closes it.
 * Errors: HGA_ERR_INVALID_ARG for an empty/out-of-range window, one that starts inside a chunk and leaves it, or
 * k_rot == k_raw with a window that is not chunk-aligned.
 */
HGA_API hga_status hga_prefill_window(const hga_params* p, const hga_buffers* buf, int64_t t_begin, int64_t t_end,
                                      void* stream);

/*
 * Instrumented hga_prefill: the same three launches groups with CUDA events recorded on `stream` between them; the
 * call synchronises `stream` and writes the elapsed milliseconds of {S0+S1 (one fused launch), S2+S3, S4} to the HOST
 * array stage_ms[3].  For measurement only (bench.py's per-stage roofline inside the real call sequence).
 */
HGA_API hga_status hga_prefill_profile(const hga_params* p, const hga_buffers* buf, void* stream, float* stage_ms_host);

/*
 * Host-buffer path.  A plan owns every device buffer of one prefill pass for `p` plus a private stream.
 * hga_host_prefill copies q/k/v from HOST memory (pinned for full speed; pageable works), runs S0..S4, copies `out`
 * (and, if non-null, group_idx [batch,n_kv_heads,seq/chunk,topk_groups] and lse) back to HOST memory and returns
 * after the stream has drained.  *_host buffers have the layouts above.  The work is pipelined over independent
 * (batch, KV head) parts on three streams, and for long sequences every part is cut into runs of whole chunks
 * (hga_prefill_window steps), so copies in, kernels and copies out overlap; results are bit-identical to hga_prefill.
 */
typedef struct hga_host_plan hga_host_plan;
HGA_API hga_status hga_host_plan_create(const hga_params* p, hga_host_plan** plan);
HGA_API hga_status hga_host_prefill(hga_host_plan* plan, const void* q_raw_host, const void* k_raw_host,
                                    const void* v_host, void* out_host, int32_t* group_idx_host, float* lse_host);
HGA_API void hga_host_plan_destroy(hga_host_plan* plan);
/* Bytes moved host->device / device->host by one hga_host_prefill call (lse/group_idx included iff requested). */
HGA_API hga_status hga_host_bytes(const hga_params* p, int32_t with_group_idx, int32_t with_lse, size_t* h2d,
                                  size_t* d2h);

#ifdef __cplusplus
}
#endif
#endif /* HGA_H_ */
