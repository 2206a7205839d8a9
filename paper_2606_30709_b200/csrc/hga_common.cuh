// Shared declarations of the CUDA path (never included by oracle/).
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "hga.h"

namespace hga {

constexpr int kChunk = 64;          // C, PAPER.md:68 ("the current implementation uses C=64")
constexpr int kMaxHalfDim = 64;     // head_dim <= 128
constexpr double kTwoPi = 6.283185307179586476925286766559;

// RoPE frequencies, computed on the host in fp64 and passed by value (theta_i = base^(-2i/D)).
struct RopeFreq {
  double turns[kMaxHalfDim];  // theta_i / (2*pi): position * turns[i] is the angle in revolutions
};

struct Derived {
  int B, N, Hq, Hkv, G, D, half;
  int C, gs, gpc;           // chunk, group, groups per chunk
  int n_b, n_g;             // chunks (= query blocks), groups per sequence
  int jb, nj;               // blocks processed by this call: [jb, jb + nj); whole sequence: 0, n_b
  long long tw0, tw1;       // token window of this call (hga_prefill_window); whole sequence: 0, N
  int F, L, L_eff, Kc, Kg;
  int n_hi_c, n_hi_g;
  long long pos0;
  long long pos_mod;  // RoPE position wrap; 0 = off
  float scale;              // softmax scale
  int fuse_q_rope;          // N2: hga_prefill does not materialise q_rot; S4 rotates its query tiles (HGA_FLAG_FUSE_Q_ROPE)
  int route_max;            // N3: block score = max over per-query scores (R19) instead of the pooled-query score
                            // (the hga_route_mode value: 1 = tensor-core prefilter where eligible, 2 = fp64 pipe only)
  bool bf16_io, bf16_out;
};

hga_status validate(const hga_params* p);
hga_status derive(const hga_params* p, Derived* d, RopeFreq* f);

#define HGA_CUDA_OK(expr)                      \
  do {                                         \
    cudaError_t _e = (expr);                   \
    if (_e != cudaSuccess) return HGA_ERR_CUDA; \
  } while (0)

// SM count of the CURRENT device (queried per call: a process may use more than one device type or MIG slice, and a
// cached static would also be a data race between concurrent callers).  Returns 0 on failure.
inline int current_sm_count() {
  int dev = 0, n = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 0;
  if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
  return n;
}

inline hga_status launch_status() { return cudaGetLastError() == cudaSuccess ? HGA_OK : HGA_ERR_CUDA; }

// ---- element I/O helpers -------------------------------------------------------------------------------------
template <typename T>
struct Io;
template <>
struct Io<float> {
  static __device__ __forceinline__ void load8(const float* p, float (&v)[8]) {
    float4 a = *reinterpret_cast<const float4*>(p), b = *reinterpret_cast<const float4*>(p + 4);
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
  }
  static __device__ __forceinline__ void store8(float* p, const float (&v)[8]) {
    *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
    *reinterpret_cast<float4*>(p + 4) = make_float4(v[4], v[5], v[6], v[7]);
  }
};
template <>
struct Io<__nv_bfloat16> {
  static __device__ __forceinline__ void load8(const __nv_bfloat16* p, float (&v)[8]) {
    uint4 r = *reinterpret_cast<const uint4*>(p);
    const uint32_t w[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      v[2 * i] = __uint_as_float(w[i] << 16);            // bf16 -> fp32 is exact
      v[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    }
  }
  static __device__ __forceinline__ void store8(__nv_bfloat16* p, const float (&v)[8]) {
    uint32_t w[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      __nv_bfloat162 h = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]);  // round-to-nearest-even, once
      w[i] = *reinterpret_cast<uint32_t*>(&h);
    }
    *reinterpret_cast<uint4*>(p) = make_uint4(w[0], w[1], w[2], w[3]);
  }
};

// ---- stage launchers (defined in the stage .cu files) --------------------------------------------------------
hga_status launch_rope(const Derived& d, const RopeFreq& f, const void* x_raw, int n_heads, void* x_rot, float* pooled,
                       cudaStream_t s);
hga_status launch_summaries(const Derived& d, const RopeFreq& f, const void* k_raw, void* k_rot, float* chunk_sum,
                            float* group_sum, cudaStream_t s);
hga_status launch_rope_summaries(const Derived& d, const RopeFreq& f, const void* q_raw, void* q_rot, float* pooled,
                                 const void* k_raw, void* k_rot, float* chunk_sum, float* group_sum, cudaStream_t s);
// rows of the score workspace per (batch, kv head) slice under the pooled-query rule: the route stage runs in slabs
constexpr int kRouteSlabRows = 1024;
inline size_t route_ws_rows(int n_b) { return (size_t)(n_b < kRouteSlabRows ? n_b : kRouteSlabRows); }
// slab_rows: 0 = kRouteSlabRows; a smaller value forces more slabs (tests)
hga_status launch_route(const Derived& d, const float* q_pooled, const float* chunk_sum, const float* group_sum,
                        int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks, int32_t* group_idx,
                        float* group_score, int32_t* n_groups, float* score_ws, cudaStream_t s, int slab_rows);
hga_status launch_route_static(const Derived& d, const float* q_pooled, const float* chunk_sum, const float* group_sum,
                               int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks, int32_t* group_idx,
                               float* group_score, int32_t* n_groups, cudaStream_t s);
size_t route_max_ws_bytes(const Derived& d);
hga_status launch_route_max(const Derived& d, const void* q_rot, const float* chunk_sum, const float* group_sum,
                            int32_t* chunk_idx, float* chunk_score, int32_t* n_chunks, int32_t* group_idx,
                            float* group_score, int32_t* n_groups, float* score_ws, cudaStream_t s);
hga_status launch_attend_simt(const Derived& d, const void* q, const void* k, const void* v, const int32_t* group_idx,
                              void* out, float* lse, cudaStream_t s);
hga_status launch_attend_tc2(const Derived& d, const void* q, const void* k, const void* v, const int32_t* group_idx,
                             void* out, float* lse, cudaStream_t s);
hga_status launch_attend_tc2_rawq(const Derived& d, const void* q_raw, const void* k, const void* v, const int32_t* group_idx,
                                  void* out, float* lse, const float2* rope_a, const float2* rope_b, cudaStream_t s);
hga_status launch_rope_tables(const Derived& d, const RopeFreq& f, float2* rope_a, float2* rope_b, cudaStream_t s);
hga_status launch_attend_pair(const Derived& d, const void* q, const void* k, const void* v, const int32_t* group_idx,
                              void* out, float* lse, cudaStream_t s);
hga_status launch_attend_tc(const Derived& d, const void* q, const void* k, const void* v, const int32_t* group_idx,
                            void* out, float* lse, cudaStream_t s);

// ---- the union key list of one (b, kv, block j) unit, as 16-token "units" -----------------------------------
// Order: sink chunks, routed groups, local chunks, current chunk.  A unit is a group of `gs`
// tokens split into 16-token pieces so that both attention kernels can treat every entry as 16 consecutive keys.
// Returns the number of 16-token pieces written to `list` (token index of the piece = list[i] * 16).
// Must be called by all threads of the CTA; ends with __syncthreads().
__device__ __forceinline__ int build_key_list(int* list, int* s_count, int j, int F, int L_eff, int gs, int Kg,
                                              const int32_t* __restrict__ gidx /* [Kg] or null */) {
  const int ppc = kChunk / 16;  // 16-token pieces per chunk
  const int ppg = gs / 16;      // pieces per group
  const int n_sink = min(F, j);
  const int loc_lo = max(max(0, j - L_eff), n_sink);  // local chunks not already covered by the sink window
  const int n_loc = max(0, j - loc_lo);
  // sink
  for (int i = threadIdx.x; i < n_sink * ppc; i += blockDim.x) list[i] = i;
  // routed: keep entries that are closed earlier groups outside the sink/local windows (set union).
  // Warp 0 compacts them in list order (ballot scan) so that the key order -- and with it the floating-point
  // summation order of the softmax -- is the same on every run.
  const int base = n_sink * ppc;
  if (threadIdx.x < 32) {
    const int lane = threadIdx.x;
    int cnt = 0;
    for (int i0 = 0; i0 < Kg; i0 += 32) {
      int i = i0 + lane;
      int g = (gidx != nullptr && i < Kg) ? gidx[i] : -1;
      bool keep = false;
      if (g >= 0) {
        int c = (g * gs) / kChunk;
        keep = (c < j) && !(c < n_sink) && !(c >= loc_lo);
      }
      unsigned m = __ballot_sync(0xffffffffu, keep);
      if (keep) {
        int slot = cnt + __popc(m & ((1u << lane) - 1u));
        for (int u = 0; u < ppg; ++u) list[base + slot * ppg + u] = g * ppg + u;
      }
      cnt += __popc(m);
    }
    if (lane == 0) *s_count = cnt;
  }
  __syncthreads();
  const int n_routed = *s_count * ppg;
  const int base2 = base + n_routed;
  for (int i = threadIdx.x; i < n_loc * ppc; i += blockDim.x) list[base2 + i] = loc_lo * ppc + i;
  const int base3 = base2 + n_loc * ppc;
  for (int i = threadIdx.x; i < ppc; i += blockDim.x) list[base3 + i] = j * ppc + i;
  __syncthreads();
  return base3 + ppc;
}

// Upper bound of build_key_list's result (host and device).
__host__ __device__ inline int max_key_pieces(int F, int L_eff, int gs, int Kg) {
  return (F + L_eff + 1) * (kChunk / 16) + Kg * (gs / 16);
}

}  // namespace hga
