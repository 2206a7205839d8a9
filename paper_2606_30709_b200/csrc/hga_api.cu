// C-ABI entry points: host-side validation and dispatch only.  All arithmetic of the path runs in the kernels.
#include <math.h>
#include <new>
#include <string.h>

#include "hga_common.cuh"

namespace hga {

static int default_n_hi(int D, double base, int span) {
  // Reading R1: pair i is "high-frequency" iff its wavelength 2*pi/theta_i is <= the span length.
  int n = 0;
  for (int i = 0; i < D / 2; ++i) {
    double theta = pow(base, -2.0 * (double)i / (double)D);
    if (kTwoPi / theta <= (double)span) ++n;
  }
  return n;
}

hga_status validate(const hga_params* p) {
  if (!p) return HGA_ERR_INVALID_ARG;
  if (p->batch <= 0 || p->seq <= 0 || p->n_q_heads <= 0 || p->n_kv_heads <= 0 || p->head_dim <= 0)
    return HGA_ERR_INVALID_ARG;
  if (p->n_q_heads % p->n_kv_heads) return HGA_ERR_INVALID_ARG;
  if (p->chunk <= 0 || p->group <= 0 || p->chunk % p->group) return HGA_ERR_INVALID_ARG;
  if (p->seq % p->chunk) return HGA_ERR_INVALID_ARG;  // only closed chunks are summarised
  if (p->n_sink < 0 || p->n_local < 0 || p->topk_chunks < 0 || p->topk_groups < 0) return HGA_ERR_INVALID_ARG;
  if (p->n_hi_chunk < -1 || p->n_hi_group < -1 || p->n_hi_chunk > p->head_dim / 2 || p->n_hi_group > p->head_dim / 2)
    return HGA_ERR_INVALID_ARG;
  if (!(p->rope_base > 0.0) || !isfinite(p->rope_base)) return HGA_ERR_INVALID_ARG;
  if (!(p->softmax_scale >= 0.0f) || !isfinite(p->softmax_scale)) return HGA_ERR_INVALID_ARG;
  if (p->io_dtype != HGA_F32 && p->io_dtype != HGA_BF16) return HGA_ERR_INVALID_ARG;
  if (p->out_dtype != HGA_F32 && p->out_dtype != HGA_BF16) return HGA_ERR_INVALID_ARG;
  if (p->attend_impl < HGA_ATTEND_AUTO || p->attend_impl > HGA_ATTEND_TCGEN05_PAIR) return HGA_ERR_INVALID_ARG;
  if (p->rope_pos_mod < 0) return HGA_ERR_INVALID_ARG;
  if (p->route_mode != HGA_ROUTE_MEAN && p->route_mode != HGA_ROUTE_MAX && p->route_mode != HGA_ROUTE_MAX_FP64)
    return HGA_ERR_INVALID_ARG;
  if (p->flags & ~(int32_t)HGA_FLAG_FUSE_Q_ROPE) return HGA_ERR_INVALID_ARG;
  if (p->rope_pos_mod > 0 && (p->rope_pos_mod % p->chunk || p->pos0 % p->chunk)) return HGA_ERR_INVALID_ARG;
  if (p->pos0 < 0 || p->pos0 + p->seq > (1ll << 40)) return HGA_ERR_INVALID_ARG;
  // what the kernels implement
  if (p->chunk != kChunk) return HGA_ERR_UNSUPPORTED;
  if (p->group % 16) return HGA_ERR_UNSUPPORTED;
  if (p->head_dim != 64 && p->head_dim != 128) return HGA_ERR_UNSUPPORTED;
  if (p->attend_impl >= HGA_ATTEND_TCGEN05 && p->io_dtype != HGA_BF16) return HGA_ERR_UNSUPPORTED;
  if ((long long)p->topk_groups * (p->group / 16) + (long long)(p->n_sink + p->n_local + 2) * 4 > 40000)
    return HGA_ERR_UNSUPPORTED;  // key list must fit in shared memory
  if ((long long)p->seq / p->chunk > 32768) return HGA_ERR_UNSUPPORTED;
  return HGA_OK;
}

hga_status derive(const hga_params* p, Derived* d, RopeFreq* f) {
  hga_status st = validate(p);
  if (st != HGA_OK) return st;
  d->B = p->batch; d->N = p->seq; d->Hq = p->n_q_heads; d->Hkv = p->n_kv_heads; d->G = p->n_q_heads / p->n_kv_heads;
  d->D = p->head_dim; d->half = p->head_dim / 2;
  d->C = p->chunk; d->gs = p->group; d->gpc = p->chunk / p->group;
  d->n_b = p->seq / p->chunk; d->n_g = p->seq / p->group;
  d->jb = 0; d->nj = d->n_b; d->tw0 = 0; d->tw1 = p->seq;
  d->F = p->n_sink; d->L = p->n_local; d->L_eff = p->n_local > 1 ? p->n_local : 1;
  d->Kc = p->topk_chunks; d->Kg = p->topk_groups;
  d->n_hi_c = p->n_hi_chunk >= 0 ? p->n_hi_chunk : default_n_hi(p->head_dim, p->rope_base, p->chunk);
  d->n_hi_g = p->n_hi_group >= 0 ? p->n_hi_group : default_n_hi(p->head_dim, p->rope_base, p->group);
  d->pos0 = p->pos0;
  d->pos_mod = p->rope_pos_mod;
  d->route_max = p->route_mode;  // 0 mean, 1 max (tensor-core prefilter where eligible), 2 max on the fp64 pipe only
  d->fuse_q_rope = (p->flags & HGA_FLAG_FUSE_Q_ROPE) ? 1 : 0;
  d->scale = p->softmax_scale > 0.0f ? p->softmax_scale : (float)(1.0 / sqrt((double)p->head_dim));
  d->bf16_io = p->io_dtype == HGA_BF16;
  d->bf16_out = p->out_dtype == HGA_BF16;
  if (f) {
    for (int i = 0; i < kMaxHalfDim; ++i) f->turns[i] = 0.0;
    for (int i = 0; i < d->half; ++i) f->turns[i] = pow(p->rope_base, -2.0 * (double)i / (double)p->head_dim) / kTwoPi;
  }
  return HGA_OK;
}

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// N2: the two RoPE tables of the fused S4 (launch_rope_tables) live behind the routing workspace
static size_t rope_tables_bytes(const Derived& d) {
  return d.fuse_q_rope ? (size_t)(d.n_b + kChunk) * d.half * sizeof(float2) : 0;
}

static size_t route_ws_bytes(const Derived& d) {
  size_t n = d.route_max ? route_max_ws_bytes(d)                               // + group-candidate scores, prefilter tables
                         : (size_t)d.B * d.Hkv * route_ws_rows(d.n_b) * d.n_b * sizeof(float);  // chunk scores, one slab
  return (n + 255) & ~(size_t)255;
}

static size_t score_ws_bytes(const Derived& d) {
  return route_ws_bytes(d) + rope_tables_bytes(d);
}

}  // namespace hga

using namespace hga;

extern "C" {

const char* hga_status_string(hga_status s) {
  switch (s) {
    case HGA_OK: return "HGA_OK";
    case HGA_ERR_INVALID_ARG: return "HGA_ERR_INVALID_ARG: null pointer, bad shape or misaligned pointer";
    case HGA_ERR_UNSUPPORTED: return "HGA_ERR_UNSUPPORTED: valid request the sm_100a kernels do not implement";
    case HGA_ERR_WORKSPACE: return "HGA_ERR_WORKSPACE: workspace missing or too small";
    case HGA_ERR_CUDA: return "HGA_ERR_CUDA: CUDA runtime or launch failure (or no device)";
  }
  return "HGA: unknown status";
}

int32_t hga_version(void) { return 100; }

int32_t hga_n_hi_rule(int32_t head_dim, double rope_base, int32_t span, int32_t rule) {
  if (head_dim <= 0 || (head_dim & 1) || !(rope_base > 0.0) || span <= 0 || rule < 0 || rule > 2) return -1;
  if (rule == 0) return default_n_hi(head_dim, rope_base, span);
  // theta_i * span >= c  <=>  i <= (D/2) * ln(span/c) / ln(base); evaluated pair by pair like the default rule
  const double c = rule == 1 ? kTwoPi * 0.5 : 1.0;
  int n = 0;
  for (int i = 0; i < head_dim / 2; ++i)
    if (pow(rope_base, -2.0 * (double)i / (double)head_dim) * (double)span >= c) ++n;
  return n;
}

int32_t hga_default_n_hi(int32_t head_dim, double rope_base, int32_t span) {
  if (head_dim <= 0 || (head_dim & 1) || !(rope_base > 0.0) || span <= 0) return -1;
  return default_n_hi(head_dim, rope_base, span);
}

hga_status hga_validate(const hga_params* p) { return validate(p); }

hga_status hga_workspace_bytes(const hga_params* p, size_t* bytes) {
  if (!bytes) return HGA_ERR_INVALID_ARG;
  Derived d;
  hga_status st = derive(p, &d, nullptr);
  if (st != HGA_OK) return st;
  *bytes = score_ws_bytes(d);
  return HGA_OK;
}

hga_status hga_rope(const hga_params* p, const void* x_raw, int32_t n_heads, void* x_rot, float* pooled,
                    void* stream) {
  Derived d;
  RopeFreq f;
  hga_status st = derive(p, &d, &f);
  if (st != HGA_OK) return st;
  if (!x_raw || !x_rot || n_heads <= 0 || !aligned16(x_raw) || !aligned16(x_rot) || !aligned16(pooled))
    return HGA_ERR_INVALID_ARG;
  if (pooled && (n_heads % d.Hkv)) return HGA_ERR_INVALID_ARG;
  return launch_rope(d, f, x_raw, n_heads, x_rot, pooled, (cudaStream_t)stream);
}

hga_status hga_build_summaries(const hga_params* p, const void* k_raw, void* k_rot, float* chunk_sum,
                               float* group_sum, void* stream) {
  Derived d;
  RopeFreq f;
  hga_status st = derive(p, &d, &f);
  if (st != HGA_OK) return st;
  if (!k_raw || !aligned16(k_raw) || !aligned16(k_rot) || !aligned16(chunk_sum) || !aligned16(group_sum))
    return HGA_ERR_INVALID_ARG;
  return launch_summaries(d, f, k_raw, k_rot, chunk_sum, group_sum, (cudaStream_t)stream);
}

hga_status hga_route(const hga_params* p, const float* q_pooled, const float* chunk_sum, const float* group_sum,
                     int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks, int32_t* group_idx, float* group_score,
                     int32_t* n_groups, void* workspace, size_t workspace_bytes, void* stream) {
  Derived d;
  hga_status st = derive(p, &d, nullptr);
  if (st != HGA_OK) return st;
  if (!q_pooled || !chunk_sum || !chunk_idx) return HGA_ERR_INVALID_ARG;
  if (d.Kg > 0 && (!group_sum || !group_idx)) return HGA_ERR_INVALID_ARG;
  if (!aligned16(q_pooled) || !aligned16(chunk_sum) || !aligned16(group_sum)) return HGA_ERR_INVALID_ARG;
  if (d.route_max) return HGA_ERR_INVALID_ARG;  // per-query scores need q_rot: hga_route_max
  if (!workspace || !aligned16(workspace) || workspace_bytes < score_ws_bytes(d)) return HGA_ERR_WORKSPACE;
  return launch_route(d, q_pooled, chunk_sum, group_sum, chunk_idx, chunk_score, n_chunks, group_idx, group_score,
                      n_groups, (float*)workspace, (cudaStream_t)stream, 0);
}

hga_status hga_route_static(const hga_params* p, const float* q_pooled, const float* chunk_sum, const float* group_sum,
                            int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks, int32_t* group_idx,
                            float* group_score, int32_t* n_groups, void* stream) {
  Derived d;
  hga_status st = derive(p, &d, nullptr);
  if (st != HGA_OK) return st;
  if (!q_pooled || !chunk_sum || !chunk_idx) return HGA_ERR_INVALID_ARG;
  if (d.Kg > 0 && (!group_sum || !group_idx)) return HGA_ERR_INVALID_ARG;
  if (!aligned16(q_pooled) || !aligned16(chunk_sum) || !aligned16(group_sum)) return HGA_ERR_INVALID_ARG;
  if (d.route_max) return HGA_ERR_INVALID_ARG;  // per-query scores need q_rot: hga_route_max
  return launch_route_static(d, q_pooled, chunk_sum, group_sum, chunk_idx, chunk_score, n_chunks, group_idx, group_score,
                             n_groups, (cudaStream_t)stream);
}

hga_status hga_route_max(const hga_params* p, const void* q_rot, const float* chunk_sum, const float* group_sum,
                         int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks, int32_t* group_idx, float* group_score,
                         int32_t* n_groups, void* workspace, size_t workspace_bytes, void* stream) {
  Derived d;
  hga_status st = derive(p, &d, nullptr);
  if (st != HGA_OK) return st;
  if (!d.route_max) return HGA_ERR_INVALID_ARG;
  if (!q_rot || !chunk_sum || !chunk_idx || !n_chunks) return HGA_ERR_INVALID_ARG;
  if (d.Kg > 0 && (!group_sum || !group_idx)) return HGA_ERR_INVALID_ARG;
  if (!aligned16(q_rot) || !aligned16(chunk_sum) || !aligned16(group_sum)) return HGA_ERR_INVALID_ARG;
  if (!workspace || !aligned16(workspace) || workspace_bytes < score_ws_bytes(d)) return HGA_ERR_WORKSPACE;
  return launch_route_max(d, q_rot, chunk_sum, group_sum, chunk_idx, chunk_score, n_chunks, group_idx, group_score,
                          n_groups, (float*)workspace, (cudaStream_t)stream);
}

static hga_status attend_blocks(const Derived& d, int impl, const void* q_rot, const void* k_rot, const void* v,
                                const int32_t* group_idx, void* out, float* lse, cudaStream_t cs) {
  hga_status st;
  if (impl == HGA_ATTEND_TCGEN05_PAIR) return launch_attend_pair(d, q_rot, k_rot, v, group_idx, out, lse, cs);
  // bf16: the persistent single-CTA kernel.  The CTA-pair kernel is correct (bit-identical results) but measured slower
  // (c5: 1.33 ms against 0.93 ms), so it is opt-in.
  if (impl == HGA_ATTEND_AUTO) impl = HGA_ATTEND_TCGEN05;
  if (impl == HGA_ATTEND_TCGEN05) {
    st = launch_attend_tc2(d, q_rot, k_rot, v, group_idx, out, lse, cs);
    if (st != HGA_ERR_UNSUPPORTED) return st;
    impl = HGA_ATTEND_TCGEN05_ITEM;
  }
  if (impl == HGA_ATTEND_TCGEN05_ITEM) return launch_attend_tc(d, q_rot, k_rot, v, group_idx, out, lse, cs);
  return launch_attend_simt(d, q_rot, k_rot, v, group_idx, out, lse, cs);
}

static hga_status attend_dispatch(const Derived& d, int impl, const void* q_rot, const void* k_rot, const void* v,
                                  const int32_t* group_idx, void* out, float* lse, cudaStream_t cs) {
  if (impl == HGA_ATTEND_AUTO && !d.bf16_io) impl = HGA_ATTEND_SIMT;
  // The tcgen05 kernels work on whole 64-row blocks.  A partial block (decode step, partial append, ragged prompt
  // tail) goes to the SIMT kernel, which masks rows and never reads a token at or past the end of the window.
  const int last = d.jb + d.nj - 1;
  const bool head_partial = d.tw0 % kChunk != 0, tail_partial = d.tw1 % kChunk != 0;
  if (head_partial) return launch_attend_simt(d, q_rot, k_rot, v, group_idx, out, lse, cs);  // one block (validated)
  if (!tail_partial) return attend_blocks(d, impl, q_rot, k_rot, v, group_idx, out, lse, cs);
  if (d.nj > 1) {
    Derived full = d;
    full.nj = d.nj - 1;
    full.tw1 = (long long)last * kChunk;
    hga_status st = attend_blocks(full, impl, q_rot, k_rot, v, group_idx, out, lse, cs);
    if (st != HGA_OK) return st;
  }
  Derived tail = d;
  tail.jb = last;
  tail.nj = 1;
  tail.tw0 = (long long)last * kChunk;
  return launch_attend_simt(tail, q_rot, k_rot, v, group_idx, out, lse, cs);
}

hga_status hga_attend(const hga_params* p, const void* q_rot, const void* k_rot, const void* v,
                      const int32_t* group_idx, void* out, float* lse, void* stream) {
  Derived d;
  hga_status st = derive(p, &d, nullptr);
  if (st != HGA_OK) return st;
  if (!q_rot || !k_rot || !v || !out) return HGA_ERR_INVALID_ARG;
  if (d.Kg > 0 && !group_idx) return HGA_ERR_INVALID_ARG;
  if (!aligned16(q_rot) || !aligned16(k_rot) || !aligned16(v) || !aligned16(out)) return HGA_ERR_INVALID_ARG;
  return attend_dispatch(d, p->attend_impl, q_rot, k_rot, v, group_idx, out, lse, (cudaStream_t)stream);
}

static hga_status prefill_impl(const hga_params* p, const hga_buffers* b, void* stream, cudaEvent_t* ev,
                               long long t_begin, long long t_end) {
  if (!b) return HGA_ERR_INVALID_ARG;
  Derived d;
  RopeFreq f;
  hga_status st = derive(p, &d, &f);
  if (st != HGA_OK) return st;
  if (t_end < 0) t_end = d.N;
  if (t_begin < 0 || t_begin >= t_end || t_end > d.N) return HGA_ERR_INVALID_ARG;
  // a window that starts inside a chunk stays inside it (one step of the active chunk)
  if (t_begin % kChunk != 0 && (t_begin / kChunk) != ((t_end - 1) / kChunk)) return HGA_ERR_INVALID_ARG;
  // In-place K (k_rot == k_raw) is only sound for chunk-aligned steps: a step that closes a chunk summarises the whole
  // 64-token tile from k_raw, and earlier partial steps would already have overwritten its first rows with rotated values.
  if (b->k_rot == b->k_raw && (t_begin % kChunk != 0 || t_end % kChunk != 0)) return HGA_ERR_INVALID_ARG;
  d.tw0 = t_begin; d.tw1 = t_end;
  d.jb = (int)(t_begin / kChunk);
  d.nj = (int)((t_end + kChunk - 1) / kChunk) - d.jb;
  const bool fuse = d.fuse_q_rope != 0;
  if (fuse) {
    // N2: whole blocks, the pooled-query rule, the persistent tcgen05 kernel (see hga_flag in hga.h)
    if (!d.bf16_io || d.route_max || t_begin % kChunk != 0 || t_end % kChunk != 0 ||
        (p->attend_impl != HGA_ATTEND_AUTO && p->attend_impl != HGA_ATTEND_TCGEN05))
      return HGA_ERR_UNSUPPORTED;
  }
  if (!b->q_raw || !b->k_raw || !b->v || (!fuse && !b->q_rot) || !b->k_rot || !b->q_pooled || !b->chunk_sum || !b->out ||
      !b->chunk_idx)
    return HGA_ERR_INVALID_ARG;
  if (d.Kg > 0 && (!b->group_sum || !b->group_idx)) return HGA_ERR_INVALID_ARG;
  if (!aligned16(b->q_raw) || !aligned16(b->q_rot) || !aligned16(b->q_pooled) || !aligned16(b->k_raw) ||
      !aligned16(b->k_rot) || !aligned16(b->chunk_sum) || !aligned16(b->group_sum) || !aligned16(b->v) ||
      !aligned16(b->out))
    return HGA_ERR_INVALID_ARG;
  if (!b->workspace || !aligned16(b->workspace) || b->workspace_bytes < score_ws_bytes(d)) return HGA_ERR_WORKSPACE;
  cudaStream_t cs = (cudaStream_t)stream;
  if (ev) HGA_CUDA_OK(cudaEventRecord(ev[0], cs));
  // S0 + S1 in one launch: the K tiles and Q tiles of a (batch, chunk) row share the position tables
  float2* rope_a = reinterpret_cast<float2*>((unsigned char*)b->workspace + route_ws_bytes(d));
  float2* rope_b = rope_a + (size_t)d.n_b * d.half;
  if (fuse) {
    st = launch_rope_tables(d, f, rope_a, rope_b, cs);
    if (st != HGA_OK) return st;
  }
  st = launch_rope_summaries(d, f, b->q_raw, fuse ? nullptr : b->q_rot, b->q_pooled, b->k_raw, b->k_rot, b->chunk_sum,
                             b->group_sum, cs);
  if (st != HGA_OK) return st;
  if (ev) HGA_CUDA_OK(cudaEventRecord(ev[1], cs));
  if (d.route_max) {
    if (t_begin % kChunk != 0 || t_end % kChunk != 0) return HGA_ERR_UNSUPPORTED;  // whole query blocks only
    if (!b->n_chunks) return HGA_ERR_INVALID_ARG;
    st = launch_route_max(d, b->q_rot, b->chunk_sum, b->group_sum, b->chunk_idx, b->chunk_score, b->n_chunks, b->group_idx,
                          b->group_score, b->n_groups, (float*)b->workspace, cs);
  } else {
    st = launch_route(d, b->q_pooled, b->chunk_sum, b->group_sum, b->chunk_idx, b->chunk_score, b->n_chunks, b->group_idx,
                      b->group_score, b->n_groups, (float*)b->workspace, cs, 0);
  }
  if (st != HGA_OK) return st;
  if (ev) HGA_CUDA_OK(cudaEventRecord(ev[2], cs));
  if (fuse) st = launch_attend_tc2_rawq(d, b->q_raw, b->k_rot, b->v, b->group_idx, b->out, b->lse, rope_a, rope_b, cs);
  else st = attend_dispatch(d, p->attend_impl, b->q_rot, b->k_rot, b->v, b->group_idx, b->out, b->lse, cs);
  if (st != HGA_OK) return st;
  if (ev) HGA_CUDA_OK(cudaEventRecord(ev[3], cs));
  return HGA_OK;
}

hga_status hga_prefill(const hga_params* p, const hga_buffers* b, void* stream) {
  return prefill_impl(p, b, stream, nullptr, 0, -1);
}

hga_status hga_prefill_window(const hga_params* p, const hga_buffers* b, int64_t t_begin, int64_t t_end, void* stream) {
  return prefill_impl(p, b, stream, nullptr, t_begin, t_end);
}

hga_status hga_prefill_profile(const hga_params* p, const hga_buffers* b, void* stream, float* stage_ms_host) {
  if (!stage_ms_host) return HGA_ERR_INVALID_ARG;
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
  hga_status st = HGA_OK;
  for (int i = 0; i < 4 && st == HGA_OK; ++i)
    if (cudaEventCreate(&ev[i]) != cudaSuccess) st = HGA_ERR_CUDA;
  if (st == HGA_OK) st = prefill_impl(p, b, stream, ev, 0, -1);
  if (st == HGA_OK && cudaEventSynchronize(ev[3]) != cudaSuccess) st = HGA_ERR_CUDA;
  for (int i = 0; i < 3 && st == HGA_OK; ++i)
    if (cudaEventElapsedTime(&stage_ms_host[i], ev[i], ev[i + 1]) != cudaSuccess) st = HGA_ERR_CUDA;
  for (int i = 0; i < 4; ++i)
    if (ev[i]) cudaEventDestroy(ev[i]);
  return st;
}

// ---------------------------------------------------------------------------------------------------------------
// Host-buffer path
// ---------------------------------------------------------------------------------------------------------------
struct hga_host_plan {
  hga_params p;
  Derived d;
  cudaStream_t stream;       // compute
  cudaStream_t s_in, s_out;  // host->device / device->host copies (PCIe is full duplex: they overlap)
  cudaEvent_t *ev_in, *ev_done;  // [n_parts]
  // the work is pipelined over parts: runs of kv_per_part KV heads of one batch item (batch_per_part == 1), or
  // batch_per_part whole batch items (kv_per_part == n_kv_heads)
  int n_parts, kv_per_part, batch_per_part;
  // every part is further cut into n_seq runs of whole chunks (hga_prefill_window steps), so that the first kernels
  // start after 1/n_seq of a part has arrived and the first results leave after 1/n_seq of its attention
  int n_seq;
  void* arena;
  size_t arena_bytes;
  hga_buffers buf;
  size_t q_bytes, kv_bytes, out_bytes, gidx_bytes, lse_bytes;
};

static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

hga_status hga_host_bytes(const hga_params* p, int32_t with_group_idx, int32_t with_lse, size_t* h2d, size_t* d2h) {
  Derived d;
  hga_status st = derive(p, &d, nullptr);
  if (st != HGA_OK) return st;
  size_t e = d.bf16_io ? 2 : 4, eo = d.bf16_out ? 2 : 4;
  size_t q = (size_t)d.B * d.Hq * d.N * d.D, kv = (size_t)d.B * d.Hkv * d.N * d.D;
  if (h2d) *h2d = (q + 2 * kv) * e;
  if (d2h)
    *d2h = q * eo + (with_group_idx ? (size_t)d.B * d.Hkv * d.n_b * d.Kg * 4 : 0) +
           (with_lse ? (size_t)d.B * d.Hq * d.N * 4 : 0);
  return HGA_OK;
}

hga_status hga_host_plan_create(const hga_params* p, hga_host_plan** out_plan) {
  if (!out_plan) return HGA_ERR_INVALID_ARG;
  *out_plan = nullptr;
  Derived d;
  hga_status st = derive(p, &d, nullptr);
  if (st != HGA_OK) return st;
  hga_host_plan* pl = new (std::nothrow) hga_host_plan();
  if (!pl) return HGA_ERR_CUDA;
  pl->p = *p;
  pl->d = d;
  size_t e = d.bf16_io ? 2 : 4, eo = d.bf16_out ? 2 : 4;
  size_t q = (size_t)d.B * d.Hq * d.N * d.D, kv = (size_t)d.B * d.Hkv * d.N * d.D;
  size_t units = (size_t)d.B * d.Hkv * d.n_b;
  pl->q_bytes = q * e; pl->kv_bytes = kv * e; pl->out_bytes = q * eo;
  pl->gidx_bytes = units * (d.Kg > 0 ? d.Kg : 1) * 4; pl->lse_bytes = (size_t)d.B * d.Hq * d.N * 4;
  size_t sizes[] = {pl->q_bytes, pl->kv_bytes, pl->kv_bytes, units * d.D * 4, units * d.D * 4,
                    (size_t)d.B * d.Hkv * d.n_g * d.D * 4, units * (d.Kc > 0 ? d.Kc : 1) * 4, pl->gidx_bytes,
                    pl->out_bytes, pl->lse_bytes, score_ws_bytes(d)};
  size_t total = 0;
  for (size_t s : sizes) total += align_up(s);
  pl->arena_bytes = total;
  if (cudaMalloc(&pl->arena, total) != cudaSuccess) { delete pl; return HGA_ERR_CUDA; }
  if (cudaStreamCreateWithFlags(&pl->stream, cudaStreamNonBlocking) != cudaSuccess) {
    cudaFree(pl->arena); delete pl; return HGA_ERR_CUDA;
  }
  // parts: units (batch, KV head) are independent in every stage and contiguous in every tensor, so the copy-in of
  // part i+1 and the copy-out of part i-1 overlap the kernels of part i.  Fewest parts >= 4 (fewer, larger parts
  // keep both the kernels and the PCIe transfers efficient).
  pl->kv_per_part = d.Hkv;
  pl->batch_per_part = 1;
  if (d.B >= 4) {
    for (int nb = d.B; nb >= 1; --nb)
      if (d.B % nb == 0 && d.B / nb >= 4) { pl->batch_per_part = nb; break; }
  } else {
    pl->kv_per_part = 1;
    for (int m = d.Hkv; m >= 1; --m)
      if (d.Hkv % m == 0 && d.B * (d.Hkv / m) >= 4) { pl->kv_per_part = m; break; }
  }
  pl->n_parts = (d.B / pl->batch_per_part) * (d.Hkv / pl->kv_per_part);
  pl->n_seq = 1;
  while (pl->n_seq < 8 && d.n_b % (2 * pl->n_seq) == 0 && d.N / (2 * pl->n_seq) >= 8192) pl->n_seq *= 2;
  const int n_ev = pl->n_parts * pl->n_seq;
  pl->ev_in = new (std::nothrow) cudaEvent_t[n_ev]();
  pl->ev_done = new (std::nothrow) cudaEvent_t[n_ev]();
  bool ok = pl->ev_in && pl->ev_done && cudaStreamCreateWithFlags(&pl->s_in, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&pl->s_out, cudaStreamNonBlocking) == cudaSuccess;
  for (int i = 0; ok && i < n_ev; ++i)
    ok = cudaEventCreateWithFlags(&pl->ev_in[i], cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&pl->ev_done[i], cudaEventDisableTiming) == cudaSuccess;
  if (!ok) { cudaFree(pl->arena); delete[] pl->ev_in; delete[] pl->ev_done; delete pl; return HGA_ERR_CUDA; }
  char* base = (char*)pl->arena;
  size_t off = 0;
  auto take = [&](size_t s) { void* r = base + off; off += align_up(s); return r; };
  hga_buffers& b = pl->buf;
  memset(&b, 0, sizeof(b));
  void* dq = take(sizes[0]); void* dk = take(sizes[1]); void* dv = take(sizes[2]);
  b.q_raw = dq; b.q_rot = dq; b.k_raw = dk; b.k_rot = dk; b.v = dv;   // RoPE in place
  b.q_pooled = (float*)take(sizes[3]); b.chunk_sum = (float*)take(sizes[4]); b.group_sum = (float*)take(sizes[5]);
  b.chunk_idx = (int32_t*)take(sizes[6]); b.group_idx = (int32_t*)take(sizes[7]);
  b.out = take(sizes[8]); b.lse = (float*)take(sizes[9]);
  b.workspace = take(sizes[10]); b.workspace_bytes = sizes[10];
  *out_plan = pl;
  return HGA_OK;
}

static hga_status host_prefill_body(hga_host_plan* pl, const void* q_host, const void* k_host, const void* v_host,
                            void* out_host, int32_t* group_idx_host, float* lse_host) {
  if (!pl || !q_host || !k_host || !v_host || !out_host) return HGA_ERR_INVALID_ARG;
  const Derived& d = pl->d;
  const int m = pl->kv_per_part, nb = pl->batch_per_part;
  hga_params sp = pl->p;  // one part: nb batch items x m KV heads (m*G query heads)
  sp.batch = nb;
  sp.n_kv_heads = m;
  sp.n_q_heads = m * d.G;
  const size_t e = d.bf16_io ? 2 : 4, eo = d.bf16_out ? 2 : 4;
  const size_t q_part = (size_t)nb * m * d.G * d.N * d.D, kv_part = (size_t)nb * m * d.N * d.D;
  const size_t unit_part = (size_t)nb * m * d.n_b;
  const size_t lse_part = (size_t)nb * m * d.G * d.N;
  auto off = [](const void* base, size_t bytes) { return (void*)((const char*)base + bytes); };
  for (int i = 0; i < pl->n_parts; ++i) {
    // parts tile every tensor contiguously: element offsets are i * part size
    const size_t qo = (size_t)i * q_part, ko = (size_t)i * kv_part, uo = (size_t)i * unit_part;
    hga_buffers b = pl->buf;
    b.q_raw = off(pl->buf.q_raw, qo * e); b.q_rot = off(pl->buf.q_rot, qo * e);
    b.k_raw = off(pl->buf.k_raw, ko * e); b.k_rot = off(pl->buf.k_rot, ko * e);
    b.v = off(pl->buf.v, ko * e);
    b.q_pooled = pl->buf.q_pooled + uo * d.D; b.chunk_sum = pl->buf.chunk_sum + uo * d.D;
    b.group_sum = pl->buf.group_sum + uo * d.gpc * d.D;
    b.chunk_idx = pl->buf.chunk_idx + uo * (d.Kc > 0 ? d.Kc : 1);
    b.group_idx = pl->buf.group_idx + uo * (d.Kg > 0 ? d.Kg : 1);
    b.out = off(pl->buf.out, qo * eo);
    b.lse = lse_host ? pl->buf.lse + (size_t)i * lse_part : nullptr;
    // the score workspace is shared: parts (and their runs) go one after another on the compute stream
    const int heads_q = nb * m * d.G, heads_kv = nb * m;
    const size_t row_in = (size_t)d.N * d.D * e, row_out = (size_t)d.N * d.D * eo;  // one head of Q/K/V, of out
    for (int c = 0; c < pl->n_seq; ++c) {
      const int ie = i * pl->n_seq + c;
      const int j0 = d.n_b / pl->n_seq * c, j1 = d.n_b / pl->n_seq * (c + 1);  // blocks of this run
      const size_t t0 = (size_t)j0 * d.C, nt = (size_t)(j1 - j0) * d.C;         // its tokens
      // rows [t0, t0 + nt) of every head: one strided copy per tensor
      HGA_CUDA_OK(cudaMemcpy2DAsync(off(b.k_raw, t0 * d.D * e), row_in, off(k_host, (ko + t0 * d.D) * e), row_in, nt * d.D * e,
                                    heads_kv, cudaMemcpyHostToDevice, pl->s_in));
      HGA_CUDA_OK(cudaMemcpy2DAsync(off(b.q_raw, t0 * d.D * e), row_in, off(q_host, (qo + t0 * d.D) * e), row_in, nt * d.D * e,
                                    heads_q, cudaMemcpyHostToDevice, pl->s_in));
      HGA_CUDA_OK(cudaMemcpy2DAsync(off(b.v, t0 * d.D * e), row_in, off(v_host, (ko + t0 * d.D) * e), row_in, nt * d.D * e,
                                    heads_kv, cudaMemcpyHostToDevice, pl->s_in));
      HGA_CUDA_OK(cudaEventRecord(pl->ev_in[ie], pl->s_in));
      HGA_CUDA_OK(cudaStreamWaitEvent(pl->stream, pl->ev_in[ie], 0));
      hga_status st = pl->n_seq == 1 ? hga_prefill(&sp, &b, (void*)pl->stream)
                                     : hga_prefill_window(&sp, &b, (int64_t)t0, (int64_t)(t0 + nt), (void*)pl->stream);
      if (st != HGA_OK) return st;
      HGA_CUDA_OK(cudaEventRecord(pl->ev_done[ie], pl->stream));
      HGA_CUDA_OK(cudaStreamWaitEvent(pl->s_out, pl->ev_done[ie], 0));
      HGA_CUDA_OK(cudaMemcpy2DAsync(off(out_host, (qo + t0 * d.D) * eo), row_out, off(b.out, t0 * d.D * eo), row_out,
                                    nt * d.D * eo, heads_q, cudaMemcpyDeviceToHost, pl->s_out));
      if (group_idx_host && d.Kg > 0)
        HGA_CUDA_OK(cudaMemcpy2DAsync(group_idx_host + (uo + j0) * d.Kg, (size_t)d.n_b * d.Kg * 4, b.group_idx + (size_t)j0 * d.Kg,
                                      (size_t)d.n_b * d.Kg * 4, (size_t)(j1 - j0) * d.Kg * 4, heads_kv, cudaMemcpyDeviceToHost,
                                      pl->s_out));
      if (lse_host)
        HGA_CUDA_OK(cudaMemcpy2DAsync(lse_host + (size_t)i * lse_part + t0, (size_t)d.N * 4, b.lse + t0, (size_t)d.N * 4, nt * 4,
                                      heads_q, cudaMemcpyDeviceToHost, pl->s_out));
    }
  }
  HGA_CUDA_OK(cudaStreamSynchronize(pl->s_out));
  HGA_CUDA_OK(cudaStreamSynchronize(pl->stream));
  return HGA_OK;
}

hga_status hga_host_prefill(hga_host_plan* pl, const void* q_host, const void* k_host, const void* v_host,
                            void* out_host, int32_t* group_idx_host, float* lse_host) {
  const hga_status st = host_prefill_body(pl, q_host, k_host, v_host, out_host, group_idx_host, lse_host);
  if (st != HGA_OK && pl) {
    // copies from / to caller-owned host buffers may still be in flight: drain them before handing control back
    cudaStreamSynchronize(pl->s_in);
    cudaStreamSynchronize(pl->stream);
    cudaStreamSynchronize(pl->s_out);
  }
  return st;
}

void hga_host_plan_destroy(hga_host_plan* pl) {
  if (!pl) return;
  for (int i = 0; i < pl->n_parts * pl->n_seq; ++i) {
    cudaEventDestroy(pl->ev_in[i]);
    cudaEventDestroy(pl->ev_done[i]);
  }
  delete[] pl->ev_in;
  delete[] pl->ev_done;
  cudaStreamDestroy(pl->s_in);
  cudaStreamDestroy(pl->s_out);
  cudaStreamDestroy(pl->stream);
  cudaFree(pl->arena);
  delete pl;
}

}  // extern "C"
