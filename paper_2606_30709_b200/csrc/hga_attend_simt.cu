// S4, fp32 SIMT kernel (Eq. (1) PAPER.md:56 restricted to the union set).
// This is the exact-arithmetic path for fp32 inputs (tcgen05 has no fp32 MMA and TF32 is too coarse for the 1e-4
// bar) and an on-device cross-check for the tensor-core kernel.  One CTA per (batch, query head, block j):
// 64 query rows against tiles of 64 gathered keys, FlashAttention-style online softmax, everything in fp32 FMA.
#include <math_constants.h>

#include "hga_common.cuh"

namespace hga {

namespace {

constexpr int kT = 256;       // threads
constexpr int kKeys = 64;     // keys per tile (4 pieces of 16 tokens)

template <typename T>
__device__ __forceinline__ float ld_as_float(const T* p);
template <>
__device__ __forceinline__ float ld_as_float<float>(const float* p) { return *p; }
template <>
__device__ __forceinline__ float ld_as_float<__nv_bfloat16>(const __nv_bfloat16* p) { return __bfloat162float(*p); }

template <typename T, typename TO, int D>
__global__ void __launch_bounds__(kT) attend_simt_kernel(const T* __restrict__ q, const T* __restrict__ k,
                                                         const T* __restrict__ v, const int32_t* __restrict__ group_idx,
                                                         TO* __restrict__ out, float* __restrict__ lse, int Hq, int Hkv, int N,
                                                         int n_b, int F, int L_eff, int gs, int Kg, float scale,
                                                         int list_cap, int jb, int tw0, int tw1) {
  constexpr int KP = D + 4;  // padded row (keeps 16-byte alignment)
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float* Qs = reinterpret_cast<float*>(smem_raw);  // [64][KP]
  float* Ks = Qs + 64 * KP;                        // [64][KP]
  float* Vs = Ks + 64 * KP;                        // [64][D]
  float* Ss = Vs + 64 * D;                         // [64][65]
  float* m_s = Ss + 64 * 65;                       // [64] running max (scaled logits)
  float* l_s = m_s + 64;                           // [64] running denominator
  float* a_s = l_s + 64;                           // [64] rescale factor of the current tile
  int* list = reinterpret_cast<int*>(a_s + 64);    // [list_cap] 16-token pieces
  __shared__ int s_count;

  const int j = jb + blockIdx.x, h = blockIdx.y, b = blockIdx.z;
  const int G = Hq / Hkv, kv = h / G;
  const int32_t* gi = group_idx ? group_idx + (((size_t)b * Hkv + kv) * n_b + j) * Kg : nullptr;
  const int n_pieces = build_key_list(list, &s_count, j, F, L_eff, gs, Kg, gi);

  const T* qbase = q + (((size_t)b * Hq + h) * N + (size_t)j * 64) * D;
  const T* kbase = k + ((size_t)b * Hkv + kv) * (size_t)N * D;
  const T* vbase = v + ((size_t)b * Hkv + kv) * (size_t)N * D;
  for (int idx = threadIdx.x; idx < 64 * D; idx += kT) {
    int r = idx / D, c = idx - r * D;
    Qs[r * KP + c] = ld_as_float(qbase + idx);
  }
  if (threadIdx.x < 64) {
    m_s[threadIdx.x] = -CUDART_INF_F;
    l_s[threadIdx.x] = 0.f;
  }
  const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
  // rows of this block inside the token window (a streaming step may cover one token): threads and warps whose rows are
  // all outside it skip the arithmetic -- a decode step then costs the gathers plus one live row, not a 64-row tile
  const int r_lo = max(0, tw0 - j * 64), r_hi = min(64, tw1 - j * 64);
  const bool thread_live = ty * 4 < r_hi && ty * 4 + 4 > r_lo;
  constexpr int OC = D / 16;  // output columns per thread
  float o[4][OC];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int c = 0; c < OC; ++c) o[a][c] = 0.f;
  __syncthreads();

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  for (int p0 = 0; p0 < n_pieces; p0 += 4) {
    const int np = min(4, n_pieces - p0);  // pieces in this tile
    // gather K, V rows (fp32 in shared memory)
    for (int idx = threadIdx.x; idx < kKeys * D; idx += kT) {
      int r = idx / D, c = idx - r * D;
      float kvv = 0.f, vv = 0.f;
      if (r < np * 16) {
        size_t tok = (size_t)list[p0 + r / 16] * 16 + (r % 16);
        if (tok < (size_t)tw1) {  // rows past the token window are not part of the cache yet (zero, never NaN)
          kvv = ld_as_float(kbase + tok * D + c);
          vv = ld_as_float(vbase + tok * D + c);
        }
      }
      Ks[r * KP + c] = kvv;
      Vs[r * D + c] = vv;
    }
    __syncthreads();
    // S = scale * Q K^T, rows 4*ty+a, cols tx+16*bcol
    {
      float acc[4][4];
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[a][c] = 0.f;
      for (int d0 = 0; thread_live && d0 < D; d0 += 4) {
        float4 qa[4], kb[4];
#pragma unroll
        for (int a = 0; a < 4; ++a) qa[a] = *reinterpret_cast<const float4*>(Qs + (ty * 4 + a) * KP + d0);
#pragma unroll
        for (int c = 0; c < 4; ++c) kb[c] = *reinterpret_cast<const float4*>(Ks + (tx + 16 * c) * KP + d0);
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            acc[a][c] = fmaf(qa[a].x, kb[c].x, acc[a][c]);
            acc[a][c] = fmaf(qa[a].y, kb[c].y, acc[a][c]);
            acc[a][c] = fmaf(qa[a].z, kb[c].z, acc[a][c]);
            acc[a][c] = fmaf(qa[a].w, kb[c].w, acc[a][c]);
          }
      }
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const int row = ty * 4 + a, col = tx + 16 * c;
          float sv = acc[a][c] * scale;
          // validity: inside the tile, and causal (key position <= query position, Eq. 1)
          bool ok = col < np * 16 && row >= r_lo && row < r_hi;
          if (ok) {
            int key_pos = list[p0 + col / 16] * 16 + (col % 16);
            ok = key_pos <= j * 64 + row;
          }
          Ss[row * 65 + col] = ok ? sv : -CUDART_INF_F;
        }
    }
    __syncthreads();
    // online softmax: warp w owns rows 8w..8w+7
    for (int rr = 0; rr < 8; ++rr) {
      const int row = warp * 8 + rr;
      if (row < r_lo || row >= r_hi) continue;  // warp-uniform
      float s0 = Ss[row * 65 + lane], s1 = Ss[row * 65 + lane + 32];
      float mx = fmaxf(s0, s1);
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, off));
      const float m_old = m_s[row];
      const float m_new = fmaxf(m_old, mx);
      const float m_use = (m_new == -CUDART_INF_F) ? 0.f : m_new;  // row fully masked so far
      const float p0v = expf(s0 - m_use), p1v = expf(s1 - m_use);   // exp(-inf) = 0
      float ps = p0v + p1v;
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) ps += __shfl_xor_sync(0xffffffffu, ps, off);
      Ss[row * 65 + lane] = p0v;
      Ss[row * 65 + lane + 32] = p1v;
      if (lane == 0) {
        const float alpha = (m_old == -CUDART_INF_F) ? 0.f : expf(m_old - m_use);
        a_s[row] = alpha;
        m_s[row] = m_new;
        l_s[row] = l_s[row] * alpha + ps;
      }
    }
    __syncthreads();
    // O = O * alpha + P V, rows 4*ty+a, cols tx+16*c
    {
      float al[4];
#pragma unroll
      for (int a = 0; a < 4; ++a) al[a] = a_s[ty * 4 + a];
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int c = 0; c < OC; ++c) o[a][c] *= al[a];
      const int nk = np * 16;
      for (int kk = 0; thread_live && kk < nk; ++kk) {
        float pv[4], vv[OC];
#pragma unroll
        for (int a = 0; a < 4; ++a) pv[a] = Ss[(ty * 4 + a) * 65 + kk];
#pragma unroll
        for (int c = 0; c < OC; ++c) vv[c] = Vs[kk * D + tx + 16 * c];
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
          for (int c = 0; c < OC; ++c) o[a][c] = fmaf(pv[a], vv[c], o[a][c]);
      }
    }
    __syncthreads();
  }
  // epilogue
  TO* obase = out + (((size_t)b * Hq + h) * N + (size_t)j * 64) * D;
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    const int row = ty * 4 + a;
    const int t_abs = j * 64 + row;
    if (t_abs < tw0 || t_abs >= tw1) continue;  // only the rows of the token window are written
    const float inv = 1.f / l_s[row];
#pragma unroll
    for (int c = 0; c < OC; ++c) {
      const float val = o[a][c] * inv;
      if constexpr (sizeof(TO) == 4) obase[(size_t)row * D + tx + 16 * c] = val;
      else obase[(size_t)row * D + tx + 16 * c] = __float2bfloat16_rn(val);
    }
  }
  if (lse != nullptr && threadIdx.x < 64 && j * 64 + (int)threadIdx.x >= tw0 && j * 64 + (int)threadIdx.x < tw1)
    lse[((size_t)b * Hq + h) * N + (size_t)j * 64 + threadIdx.x] = m_s[threadIdx.x] + logf(l_s[threadIdx.x]);
}

// A few query rows of one block (single-token decode, a short append): one CTA per (batch, query head), the key
// list split over 8 warps that each run an online softmax over their keys (a lane holds D/32 dimensions of q, o and
// of every key / value row; one warp-wide dot product per key), then the 8 partial (m, l, o) results are merged.
// Same arithmetic as the tile kernel above (fp32, exact causal rule), without its 64-row tile.
template <typename T, typename TO, int D>
__global__ void __launch_bounds__(256) attend_rows_kernel(const T* __restrict__ q, const T* __restrict__ k,
                                                          const T* __restrict__ v, const int32_t* __restrict__ group_idx,
                                                          TO* __restrict__ out, float* __restrict__ lse, int Hq, int Hkv, int N,
                                                          int n_b, int F, int L_eff, int gs, int Kg, float scale, int list_cap,
                                                          int j, int tw0, int tw1) {
  constexpr int DL = D / 32, NWARP = 8;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float* part = reinterpret_cast<float*>(smem_raw);      // [NWARP][D + 2]: o, m, l
  int* list = reinterpret_cast<int*>(part + NWARP * (D + 2));  // [list_cap] 16-token pieces
  __shared__ int s_count;
  const int h = blockIdx.x, b = blockIdx.y;
  const int G = Hq / Hkv, kv = h / G;
  const int32_t* gi = group_idx ? group_idx + (((size_t)b * Hkv + kv) * n_b + j) * Kg : nullptr;
  const int n_keys = build_key_list(list, &s_count, j, F, L_eff, gs, Kg, gi) * 16;
  const T* kbase = k + ((size_t)b * Hkv + kv) * (size_t)N * D;
  const T* vbase = v + ((size_t)b * Hkv + kv) * (size_t)N * D;
  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const int r_lo = max(0, tw0 - j * 64), r_hi = min(64, tw1 - j * 64);
  for (int r = r_lo; r < r_hi; ++r) {
    const int t_abs = j * 64 + r;
    const T* qrow = q + (((size_t)b * Hq + h) * N + (size_t)t_abs) * D + lane * DL;
    float qv[DL], o[DL];
#pragma unroll
    for (int u = 0; u < DL; ++u) {
      qv[u] = ld_as_float(qrow + u) * scale;
      o[u] = 0.f;
    }
    float m = -CUDART_INF_F, l = 0.f;
    for (int kidx = warp; kidx < n_keys; kidx += NWARP) {
      const int tok = list[kidx / 16] * 16 + (kidx % 16);
      if (tok > t_abs || tok >= tw1) continue;  // causal (Eq. 1); warp-uniform
      const T* krow = kbase + (size_t)tok * D + lane * DL;
      const T* vrow = vbase + (size_t)tok * D + lane * DL;
      float sdot = 0.f, vv[DL];
#pragma unroll
      for (int u = 0; u < DL; ++u) {
        sdot = fmaf(qv[u], ld_as_float(krow + u), sdot);
        vv[u] = ld_as_float(vrow + u);
      }
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) sdot += __shfl_xor_sync(0xffffffffu, sdot, off);
      const float m_new = fmaxf(m, sdot);
      const float alpha = expf(m - m_new), pw = expf(sdot - m_new);  // exp(-inf) = 0 on the first key
      l = l * alpha + pw;
#pragma unroll
      for (int u = 0; u < DL; ++u) o[u] = fmaf(pw, vv[u], o[u] * alpha);
      m = m_new;
    }
    float* pr = part + warp * (D + 2);
#pragma unroll
    for (int u = 0; u < DL; ++u) pr[lane * DL + u] = o[u];
    if (lane == 0) {
      pr[D] = m;
      pr[D + 1] = l;
    }
    __syncthreads();
    if (warp == 0) {
      float M = -CUDART_INF_F;
#pragma unroll
      for (int w = 0; w < NWARP; ++w) M = fmaxf(M, part[w * (D + 2) + D]);  // finite: the row's own key is always there
      float L = 0.f, acc[DL];
#pragma unroll
      for (int u = 0; u < DL; ++u) acc[u] = 0.f;
#pragma unroll
      for (int w = 0; w < NWARP; ++w) {
        const float wgt = expf(part[w * (D + 2) + D] - M);  // 0 for a warp that saw no key
        L = fmaf(part[w * (D + 2) + D + 1], wgt, L);
#pragma unroll
        for (int u = 0; u < DL; ++u) acc[u] = fmaf(part[w * (D + 2) + lane * DL + u], wgt, acc[u]);
      }
      TO* orow = out + (((size_t)b * Hq + h) * N + (size_t)t_abs) * D + lane * DL;
      const float inv = 1.f / L;
#pragma unroll
      for (int u = 0; u < DL; ++u) {
        if constexpr (sizeof(TO) == 4) orow[u] = acc[u] * inv;
        else orow[u] = __float2bfloat16_rn(acc[u] * inv);
      }
      if (lse != nullptr && lane == 0) lse[((size_t)b * Hq + h) * N + (size_t)t_abs] = M + logf(L);
    }
    __syncthreads();
  }
}

template <typename T, typename TO, int D>
hga_status launch_t(const Derived& d, const void* q, const void* k, const void* v, const int32_t* gi, void* out, float* lse,
                    cudaStream_t s) {
  const int list_cap = max_key_pieces(d.F, d.L_eff, d.gs, d.Kg);
  const long long live_rows = d.tw1 - (d.tw0 > (long long)d.jb * 64 ? d.tw0 : (long long)d.jb * 64);
  if (d.nj == 1 && live_rows <= 4) {  // decode / short append: no 64-row tile
    const size_t smem_r = sizeof(float) * 8 * (D + 2) + sizeof(int) * (size_t)list_cap;
    if (smem_r > 200 * 1024) return HGA_ERR_UNSUPPORTED;
    auto kern_r = attend_rows_kernel<T, TO, D>;
    HGA_CUDA_OK(cudaFuncSetAttribute(kern_r, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_r));
    kern_r<<<dim3(d.Hq, d.B), 256, smem_r, s>>>((const T*)q, (const T*)k, (const T*)v, gi, (TO*)out, lse, d.Hq, d.Hkv, d.N, d.n_b,
                                                d.F, d.L_eff, d.gs, d.Kg, d.scale, list_cap, d.jb, (int)d.tw0, (int)d.tw1);
    return launch_status();
  }
  const size_t smem = sizeof(float) * (2 * 64 * (D + 4) + 64 * D + 64 * 65 + 3 * 64) + sizeof(int) * (size_t)list_cap;
  if (smem > 220 * 1024) return HGA_ERR_UNSUPPORTED;
  auto kern = attend_simt_kernel<T, TO, D>;
  HGA_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  dim3 grid(d.nj, d.Hq, d.B);
  kern<<<grid, kT, smem, s>>>((const T*)q, (const T*)k, (const T*)v, gi, (TO*)out, lse, d.Hq, d.Hkv, d.N, d.n_b, d.F,
                              d.L_eff, d.gs, d.Kg, d.scale, list_cap, d.jb, (int)d.tw0, (int)d.tw1);
  return launch_status();
}

template <typename T, typename TO>
hga_status launch_d(const Derived& d, const void* q, const void* k, const void* v, const int32_t* gi, void* out, float* lse,
                    cudaStream_t s) {
  return d.D == 128 ? launch_t<T, TO, 128>(d, q, k, v, gi, out, lse, s) : launch_t<T, TO, 64>(d, q, k, v, gi, out, lse, s);
}

}  // namespace

hga_status launch_attend_simt(const Derived& d, const void* q, const void* k, const void* v, const int32_t* group_idx,
                              void* out, float* lse, cudaStream_t s) {
  if (d.bf16_io) {
    return d.bf16_out ? launch_d<__nv_bfloat16, __nv_bfloat16>(d, q, k, v, group_idx, out, lse, s)
                      : launch_d<__nv_bfloat16, float>(d, q, k, v, group_idx, out, lse, s);
  }
  return d.bf16_out ? launch_d<float, __nv_bfloat16>(d, q, k, v, group_idx, out, lse, s)
                    : launch_d<float, float>(d, q, k, v, group_idx, out, lse, s);
}

}  // namespace hga
