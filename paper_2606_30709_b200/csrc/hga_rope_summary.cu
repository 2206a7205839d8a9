// S0 (RoPE on Q + pooled block query) and S1 (RoPE on K + mixed-RoPE chunk/group summaries).
// Both are one pass over their tensor: HBM-bound, 16-byte vector loads/stores, one CTA per 64-token chunk and a
// few heads.  PAPER.md:62 (RoPE), 80-89 (summaries), 33/45/97 (chunk-shared per-KV-head routing query).
//
// Numerics: the angle p*theta_i is reduced in fp64 (revolutions -> fractional part), the reduced angle is split
// into an fp32 head and tail, sincosf() is taken on the head and corrected to first order with the tail, so
// cos/sin carry ~1 ulp(fp32) error at any position.  The rotation is fp32 FMA; every mean is accumulated in fp64
// from the un-rounded fp32 values and rounded once to float; the rotated tensor is rounded once to io_dtype.
#include "hga_common.cuh"

namespace hga {

namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ double reduced_angle(double pos, double turns) {
  double u = pos * turns;  // revolutions
  double fr = u - rint(u);  // [-0.5, 0.5]
  return fr * kTwoPi;
}

__device__ __forceinline__ float2 cos_sin_f32(double pos, double turns) {
  double ang = reduced_angle(pos, turns);
  float ah = (float)ang;
  float al = (float)(ang - (double)ah);
  float sh, ch;
  sincosf(ah, &sh, &ch);
  return make_float2(fmaf(-sh, al, ch), fmaf(ch, al, sh));
}

// cs[t * half + i] = (cos, sin)((pos_first + t) * theta_i) for the chunk's 64 tokens.
__device__ __forceinline__ void fill_table(float2* cs, const RopeFreq& f, int half, long long pos_first) {
  for (int idx = threadIdx.x; idx < kChunk * half; idx += blockDim.x) {
    int t = idx / half, i = idx - t * half;
    cs[idx] = cos_sin_f32((double)(pos_first + t), f.turns[i]);
  }
}

// ----------------------------------------------------------------------------------------------------------------
// S0: x_rot = RoPE(x_raw); pooled = mean over (chunk tokens, heads of the pool group) of the rotated vectors.
// grid (n_b, n_heads / heads_per_cta, B); heads_per_cta is a multiple of pool_heads.
// ----------------------------------------------------------------------------------------------------------------
template <typename T, int D>
__global__ void __launch_bounds__(kThreads) rope_pool_kernel(const __grid_constant__ RopeFreq f,
                                                             const T* x_raw, T* x_rot,  // may alias (in-place RoPE)
                                                            
                                                             float* __restrict__ pooled, int n_heads, int N, int n_b,
                                                             int heads_per_cta, int pool_heads, long long pos0) {
  constexpr int half = D / 2;
  constexpr int OCT = D / 16;               // threads per token (8 pairs each)
  constexpr int TOK_PER_PASS = kThreads / OCT;
  constexpr int PASSES = kChunk / TOK_PER_PASS;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* cs = reinterpret_cast<float2*>(smem_raw);                              // [64][half]
  double* red = reinterpret_cast<double*>(smem_raw + sizeof(float2) * kChunk * half);  // [TOK_PER_PASS][D]

  const int j = blockIdx.x, b = blockIdx.z;
  const int head0 = blockIdx.y * heads_per_cta;
  fill_table(cs, f, half, pos0 + (long long)j * kChunk);
  __syncthreads();

  const int oct = threadIdx.x % OCT, slot = threadIdx.x / OCT;
  const int i0 = oct * 8;
  double acc[16];
#pragma unroll
  for (int u = 0; u < 16; ++u) acc[u] = 0.0;

  for (int hh = 0; hh < heads_per_cta; ++hh) {
    const int h = head0 + hh;
    const size_t row0 = ((size_t)b * n_heads + h) * N + (size_t)j * kChunk;
#pragma unroll
    for (int ps = 0; ps < PASSES; ++ps) {
      const int t = ps * TOK_PER_PASS + slot;
      const T* src = x_raw + (row0 + t) * D;
      float a[8], bb[8], ra[8], rb[8];
      Io<T>::load8(src + i0, a);
      Io<T>::load8(src + half + i0, bb);
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        float2 c = cs[t * half + i0 + u];
        ra[u] = fmaf(a[u], c.x, -(bb[u] * c.y));
        rb[u] = fmaf(bb[u], c.x, a[u] * c.y);
        acc[u] += (double)ra[u];
        acc[8 + u] += (double)rb[u];
      }
      T* dst = x_rot + (row0 + t) * D;
      Io<T>::store8(dst + i0, ra);
      Io<T>::store8(dst + half + i0, rb);
    }
    if (pooled != nullptr && (hh + 1) % pool_heads == 0) {
      // cross-thread reduction over the TOK_PER_PASS token slots, fixed order -> deterministic
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        red[slot * D + i0 + u] = acc[u];
        red[slot * D + half + i0 + u] = acc[8 + u];
        acc[u] = 0.0;
        acc[8 + u] = 0.0;
      }
      __syncthreads();
      if (threadIdx.x < D) {
        double s = 0.0;
        for (int q = 0; q < TOK_PER_PASS; ++q) s += red[q * D + threadIdx.x];
        const int pg = h / pool_heads;  // pool group index == kv head
        const int n_pg = n_heads / pool_heads;
        pooled[(((size_t)b * n_pg + pg) * n_b + j) * D + threadIdx.x] = (float)(s / (double)(pool_heads * kChunk));
      }
      __syncthreads();
    }
  }
}

// ----------------------------------------------------------------------------------------------------------------
// S1: k_rot = RoPE(k_raw); chunk and group summaries by the mixed rule.
// grid (n_b, Hkv / heads_per_cta, B)
// ----------------------------------------------------------------------------------------------------------------
template <typename T, int D>
__global__ void __launch_bounds__(kThreads) summaries_kernel(const __grid_constant__ RopeFreq f,
                                                             const T* k_raw, T* k_rot,  // may alias (in-place RoPE)
                                                            
                                                             float* __restrict__ chunk_sum, float* __restrict__ group_sum,
                                                             int Hkv, int N, int n_b, int heads_per_cta, int gs,
                                                             int n_hi_c, int n_hi_g, long long pos0) {
  constexpr int half = D / 2;
  constexpr int OCT = D / 16;
  constexpr int TOK_PER_PASS = kThreads / OCT;
  constexpr int PASSES = kChunk / TOK_PER_PASS;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* cs = reinterpret_cast<float2*>(smem_raw);                    // [64][half]
  float* rot_s = reinterpret_cast<float*>(cs + kChunk * half);         // [64][D] rotated keys (fp32, un-rounded)
  float* raw_s = rot_s + kChunk * D;                                   // [64][D] raw keys
  double2* mid_g = reinterpret_cast<double2*>(raw_s + kChunk * D);     // [gpc][half] (cos, sin) at group middles
  double2* mid_c = mid_g + (kChunk / 16) * half;                       // [half]      (cos, sin) at the chunk middle
  double* dsum = reinterpret_cast<double*>(mid_c + half);              // [gpc][4][half]

  const int j = blockIdx.x, b = blockIdx.z;
  const int head0 = blockIdx.y * heads_per_cta;
  const int gpc = kChunk / gs;
  const long long pos_first = pos0 + (long long)j * kChunk;
  fill_table(cs, f, half, pos_first);
  // middle positions (reading R2: start + (S-1)/2), full fp64 sincos -- once per CTA
  for (int idx = threadIdx.x; idx < (gpc + 1) * half; idx += blockDim.x) {
    int g = idx / half, i = idx - g * half;
    double pm = (g < gpc) ? (double)pos_first + (double)(g * gs) + 0.5 * (double)(gs - 1)
                          : (double)pos_first + 0.5 * (double)(kChunk - 1);
    double s, c;
    sincos(reduced_angle(pm, f.turns[i]), &s, &c);
    if (g < gpc) mid_g[g * half + i] = make_double2(c, s);
    else mid_c[i] = make_double2(c, s);
  }
  __syncthreads();

  const int oct = threadIdx.x % OCT, slot = threadIdx.x / OCT;
  const int i0 = oct * 8;
  // phase-B role: thread (g, i) sums group g, pair i
  const int bg = threadIdx.x / half, bi = threadIdx.x % half;
  const bool b_active = bg < gpc;

  for (int hh = 0; hh < heads_per_cta; ++hh) {
    const int h = head0 + hh;
    const size_t row0 = ((size_t)b * Hkv + h) * N + (size_t)j * kChunk;
    // phase A: rotate, store, stage rotated + raw values in shared memory
#pragma unroll
    for (int ps = 0; ps < PASSES; ++ps) {
      const int t = ps * TOK_PER_PASS + slot;
      const T* src = k_raw + (row0 + t) * D;
      float a[8], bb[8], ra[8], rb[8];
      Io<T>::load8(src + i0, a);
      Io<T>::load8(src + half + i0, bb);
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        float2 c = cs[t * half + i0 + u];
        ra[u] = fmaf(a[u], c.x, -(bb[u] * c.y));
        rb[u] = fmaf(bb[u], c.x, a[u] * c.y);
      }
      if (k_rot != nullptr) {
        T* dst = k_rot + (row0 + t) * D;
        Io<T>::store8(dst + i0, ra);
        Io<T>::store8(dst + half + i0, rb);
      }
      float* pr = rot_s + t * D;
      float* pw = raw_s + t * D;
      *reinterpret_cast<float4*>(pr + i0) = make_float4(ra[0], ra[1], ra[2], ra[3]);
      *reinterpret_cast<float4*>(pr + i0 + 4) = make_float4(ra[4], ra[5], ra[6], ra[7]);
      *reinterpret_cast<float4*>(pr + half + i0) = make_float4(rb[0], rb[1], rb[2], rb[3]);
      *reinterpret_cast<float4*>(pr + half + i0 + 4) = make_float4(rb[4], rb[5], rb[6], rb[7]);
      *reinterpret_cast<float4*>(pw + i0) = make_float4(a[0], a[1], a[2], a[3]);
      *reinterpret_cast<float4*>(pw + i0 + 4) = make_float4(a[4], a[5], a[6], a[7]);
      *reinterpret_cast<float4*>(pw + half + i0) = make_float4(bb[0], bb[1], bb[2], bb[3]);
      *reinterpret_cast<float4*>(pw + half + i0 + 4) = make_float4(bb[4], bb[5], bb[6], bb[7]);
    }
    __syncthreads();
    // phase B: per (group, pair) sums in fp64, fixed order
    if (b_active) {
      double ra = 0.0, rb = 0.0, wa = 0.0, wb = 0.0;
      for (int t = bg * gs; t < (bg + 1) * gs; ++t) {
        ra += (double)rot_s[t * D + bi];
        rb += (double)rot_s[t * D + half + bi];
        wa += (double)raw_s[t * D + bi];
        wb += (double)raw_s[t * D + half + bi];
      }
      dsum[(bg * 4 + 0) * half + bi] = ra;
      dsum[(bg * 4 + 1) * half + bi] = rb;
      dsum[(bg * 4 + 2) * half + bi] = wa;
      dsum[(bg * 4 + 3) * half + bi] = wb;
      if (group_sum != nullptr) {
        double sa, sb;
        const double inv = 1.0 / (double)gs;
        if (bi < n_hi_g) {  // high-frequency pair: rotate per token, then average
          sa = ra * inv;
          sb = rb * inv;
        } else {            // low-frequency pair: average raw keys, rotate at the middle position
          double2 m = mid_g[bg * half + bi];
          double ma = wa * inv, mb = wb * inv;
          sa = ma * m.x - mb * m.y;
          sb = mb * m.x + ma * m.y;
        }
        float* dst = group_sum + (((size_t)b * Hkv + h) * (size_t)(n_b * gpc) + (size_t)j * gpc + bg) * D;
        dst[bi] = (float)sa;
        dst[half + bi] = (float)sb;
      }
    }
    __syncthreads();
    if (chunk_sum != nullptr && threadIdx.x < half) {
      const int i = threadIdx.x;
      double ra = 0.0, rb = 0.0, wa = 0.0, wb = 0.0;
      for (int g = 0; g < gpc; ++g) {
        ra += dsum[(g * 4 + 0) * half + i];
        rb += dsum[(g * 4 + 1) * half + i];
        wa += dsum[(g * 4 + 2) * half + i];
        wb += dsum[(g * 4 + 3) * half + i];
      }
      const double inv = 1.0 / (double)kChunk;
      double sa, sb;
      if (i < n_hi_c) {
        sa = ra * inv;
        sb = rb * inv;
      } else {
        double2 m = mid_c[i];
        double ma = wa * inv, mb = wb * inv;
        sa = ma * m.x - mb * m.y;
        sb = mb * m.x + ma * m.y;
      }
      float* dst = chunk_sum + (((size_t)b * Hkv + h) * n_b + j) * D;
      dst[i] = (float)sa;
      dst[half + i] = (float)sb;
    }
    // The next head's phase A only writes rot_s/raw_s (phase B readers are past the barrier above); its phase B
    // writes dsum only after the next __syncthreads(), which the finalising threads also reach.
  }
}

// Largest divisor hpc of n_items (a multiple of `quantum`) that still leaves >= target CTAs.
int pick_per_cta(int n_items, int quantum, long long other_ctas, long long target) {
  int best = quantum;
  for (int hpc = quantum; hpc <= n_items; hpc += quantum) {
    if (n_items % hpc) continue;
    if (other_ctas * (n_items / hpc) >= target) best = hpc;
  }
  return best;
}

template <typename T, int D>
hga_status launch_rope_t(const Derived& d, const RopeFreq& f, const void* x_raw, int n_heads, void* x_rot, float* pooled,
                         cudaStream_t s) {
  const int pool_heads = pooled ? n_heads / d.Hkv : 1;
  const int hpc = pick_per_cta(n_heads, pool_heads, (long long)d.n_b * d.B, 1024);
  const size_t smem = sizeof(float2) * kChunk * (D / 2) + sizeof(double) * (kThreads / (D / 16)) * D;
  auto kern = rope_pool_kernel<T, D>;
  HGA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  dim3 grid(d.n_b, n_heads / hpc, d.B);
  kern<<<grid, kThreads, smem, s>>>(f, (const T*)x_raw, (T*)x_rot, pooled, n_heads, d.N, d.n_b, hpc, pool_heads, d.pos0);
  return launch_status();
}

template <typename T, int D>
hga_status launch_summaries_t(const Derived& d, const RopeFreq& f, const void* k_raw, void* k_rot, float* chunk_sum,
                              float* group_sum, cudaStream_t s) {
  const int hpc = pick_per_cta(d.Hkv, 1, (long long)d.n_b * d.B, 1024);
  constexpr int half = D / 2;
  const size_t smem = sizeof(float2) * kChunk * half + 2 * sizeof(float) * kChunk * D +
                      sizeof(double2) * ((kChunk / 16) + 1) * half + sizeof(double) * (kChunk / 16) * 4 * half;
  auto kern = summaries_kernel<T, D>;
  HGA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  dim3 grid(d.n_b, d.Hkv / hpc, d.B);
  kern<<<grid, kThreads, smem, s>>>(f, (const T*)k_raw, (T*)k_rot, chunk_sum, group_sum, d.Hkv, d.N, d.n_b, hpc, d.gs,
                                    d.n_hi_c, d.n_hi_g, d.pos0);
  return launch_status();
}

}  // namespace

hga_status launch_rope(const Derived& d, const RopeFreq& f, const void* x_raw, int n_heads, void* x_rot, float* pooled,
                       cudaStream_t s) {
  if (d.bf16_io) {
    return d.D == 128 ? launch_rope_t<__nv_bfloat16, 128>(d, f, x_raw, n_heads, x_rot, pooled, s)
                      : launch_rope_t<__nv_bfloat16, 64>(d, f, x_raw, n_heads, x_rot, pooled, s);
  }
  return d.D == 128 ? launch_rope_t<float, 128>(d, f, x_raw, n_heads, x_rot, pooled, s)
                    : launch_rope_t<float, 64>(d, f, x_raw, n_heads, x_rot, pooled, s);
}

hga_status launch_summaries(const Derived& d, const RopeFreq& f, const void* k_raw, void* k_rot, float* chunk_sum,
                            float* group_sum, cudaStream_t s) {
  if (d.bf16_io) {
    return d.D == 128 ? launch_summaries_t<__nv_bfloat16, 128>(d, f, k_raw, k_rot, chunk_sum, group_sum, s)
                      : launch_summaries_t<__nv_bfloat16, 64>(d, f, k_raw, k_rot, chunk_sum, group_sum, s);
  }
  return d.D == 128 ? launch_summaries_t<float, 128>(d, f, k_raw, k_rot, chunk_sum, group_sum, s)
                    : launch_summaries_t<float, 64>(d, f, k_raw, k_rot, chunk_sum, group_sum, s);
}

}  // namespace hga
