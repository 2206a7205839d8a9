// The online-softmax step of the tcgen05 attention kernels (attend_tc2_kernel, attend_pair_kernel): one thread owns
// one query row of a 128-row tile; S (fp32, 128 key columns) is read from TMEM, P (bf16) is written over it.
// Arithmetic: fp32, base 2 (scores scaled by scale * log2 e), running max refreshed lazily (only when it grows by
// more than 2^8, which leaves the result mathematically unchanged), packed FFMA2 / FADD2, FMNMX3 row max.
#pragma once

#include <math_constants.h>

#include <type_traits>

#include "hga_tc_ptx.cuh"

namespace hga {
namespace tc {

constexpr float kRescaleThreshold = 8.0f;  // log2 units

// compile-time experiment knobs (never set in a product build)
#ifndef HGA_S4_EMU_PERIOD
#define HGA_S4_EMU_PERIOD 4
#endif
#ifndef HGA_S4_EMU_COUNT
#define HGA_S4_EMU_COUNT 0  // exp2 on the FMA pipe for pairs p with (p % PERIOD) < COUNT
#endif
#ifndef HGA_S4_DIAG
#define HGA_S4_DIAG 0  // bit mask: 1 = no softmax arithmetic, 2 = no MMAs, 4 = no MUFU, 8 = no K/V TMA
#endif
constexpr int kDiag = HGA_S4_DIAG;
constexpr int kEmuPeriod = HGA_S4_EMU_PERIOD;
constexpr int kEmuCount = HGA_S4_EMU_COUNT;

// exp2(x) for x <= ~8 evaluated without MUFU: n = round(x), r = x - n in [-0.5, 0.5], 2^r by a degree-3 polynomial
// (weighted least squares on Chebyshev nodes, max rel. error 7.5e-5), exponent added in the integer domain.
__device__ __forceinline__ void exp2_poly2(float x0, float x1, float& p0, float& p1) {
  const float kMagic = 12582912.0f;  // 1.5 * 2^23: adding it rounds to the nearest integer in the low mantissa bits
  x0 = fmaxf(x0, -125.0f);
  x1 = fmaxf(x1, -125.0f);
  const uint64_t x = pack2(x0, x1);
  const uint64_t magic = pack2(kMagic, kMagic);
  const uint64_t t = add2(x, magic);
  const uint64_t nf = add2(t, pack2(-kMagic, -kMagic));
  const uint64_t r = fma2(nf, pack2(-1.0f, -1.0f), x);
  uint64_t p = fma2(pack2(0.0551716648042202f, 0.0551716648042202f), r, pack2(0.2426111251115799f, 0.2426111251115799f));
  p = fma2(p, r, pack2(0.6932609677314758f, 0.6932609677314758f));
  p = fma2(p, r, pack2(0.9999280571937561f, 0.9999280571937561f));
  float t0, t1, q0, q1;
  unpack2(t, t0, t1);
  unpack2(p, q0, q1);
  p0 = __uint_as_float(__float_as_uint(q0) + (__float_as_uint(t0) << 23));
  p1 = __uint_as_float(__float_as_uint(q1) + (__float_as_uint(t1) << 23));
}

// One key tile of one query row.
//   s_addr / o_addr : TMEM addresses (this warp's lane quadrant) of S_t / O_t;  D: head_dim (columns of O_t)
//   causal          : key column c (< 64) is token c of the row's own chunk; row index in the chunk is r64
//   nk              : valid key columns of the tile (a multiple of 16; 128 = full tile)
//   o_live          : O_t already holds partial sums (not the first tile of its accumulator)
//   arrive_a / _b   : called by every lane once keys 0..63 / 64..127 of P are in TMEM (tcgen05.wait::st and the
//                     before_thread_sync fence have been issued; the callee does the warp-level arrive)
template <int D, class ArriveA, class ArriveB>
__device__ __forceinline__ void softmax_tile(uint32_t s_addr, uint32_t o_addr, bool causal, int r64, int nk, bool o_live,
                                             float sl2, float& m_run, float& l_run, ArriveA arrive_a, ArriveB arrive_b,
                                             long long* tr = nullptr) {
#ifdef HGA_S4_TRACE
#define HGA_TR(e) do { if (tr != nullptr && (threadIdx.x & 31) == 0) tr[e] = clock64(); } while (0)
#else
#define HGA_TR(e) do { } while (0)
#endif
  const uint64_t sl2x2 = pack2(sl2, sl2);
  uint32_t sr[128];
  tmem_ld32(s_addr + 0, sr + 0);
  tmem_ld32(s_addr + 32, sr + 32);
  tmem_ld32(s_addr + 64, sr + 64);
  tmem_ld32(s_addr + 96, sr + 96);
  tmem_wait_ld();
  HGA_TR(1);
  if (causal) {
#pragma unroll
    for (int c = 1; c < 64; ++c)
      if (c > r64) sr[c] = __float_as_uint(-CUDART_INF_F);
  }
  if (nk < 128) {
#pragma unroll
    for (int c = 16; c < 128; ++c)
      if (c >= nk) sr[c] = __float_as_uint(-CUDART_INF_F);
  }
  float mx0 = max3(__uint_as_float(sr[0]), __uint_as_float(sr[1]), __uint_as_float(sr[2]));
  float mx1 = max3(__uint_as_float(sr[3]), __uint_as_float(sr[4]), __uint_as_float(sr[5]));
  float mx2 = max3(__uint_as_float(sr[6]), __uint_as_float(sr[7]), __uint_as_float(sr[8]));
  float mx3 = max3(__uint_as_float(sr[9]), __uint_as_float(sr[10]), __uint_as_float(sr[11]));
#pragma unroll
  for (int c = 12; c < 124; c += 8) {
    mx0 = max3(mx0, __uint_as_float(sr[c]), __uint_as_float(sr[c + 1]));
    mx1 = max3(mx1, __uint_as_float(sr[c + 2]), __uint_as_float(sr[c + 3]));
    mx2 = max3(mx2, __uint_as_float(sr[c + 4]), __uint_as_float(sr[c + 5]));
    mx3 = max3(mx3, __uint_as_float(sr[c + 6]), __uint_as_float(sr[c + 7]));
  }
  mx0 = max3(mx0, __uint_as_float(sr[124]), __uint_as_float(sr[125]));
  mx1 = max3(mx1, __uint_as_float(sr[126]), __uint_as_float(sr[127]));
  const float m_new = fmaxf(m_run, fmaxf(max3(mx0, mx1, mx2), mx3));
  const bool need = (m_new - m_run) * sl2 > kRescaleThreshold;  // first tile: +inf > 8
  if (__any_sync(0xffffffffu, need)) {
    float alpha = 1.f;
    if (need) {
      alpha = (m_run == -CUDART_INF_F) ? 0.f : fast_exp2((m_run - m_new) * sl2);
      m_run = m_new;
      l_run *= alpha;
    }
    if (o_live) {
      // O_t is quiescent here: S_FULL of this tile was committed after the previous P V of the accumulator
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        uint32_t orr[32];
        tmem_ld32(o_addr + c0, orr);
        tmem_wait_ld();
#pragma unroll
        for (int c = 0; c < 32; ++c) orr[c] = __float_as_uint(__uint_as_float(orr[c]) * alpha);
        tmem_st32(o_addr + c0, orr);
      }
    }
  }
  HGA_TR(2);
  const float neg_m = -m_run * sl2;  // finite: the diagonal key of tile 0 is never masked
  const uint64_t negm2 = pack2(neg_m, neg_m);
  uint64_t acc0 = pack2(0.f, 0.f), acc1 = acc0;
#pragma unroll
  for (int c0 = 0; c0 < 128; c0 += 32) {
    uint32_t pr[16];
#pragma unroll
    for (int c = 0; c < 16; ++c) {
      const int pi = (c0 / 2 + c);  // pair index 0..63
      const uint64_t x = fma2(pack2(__uint_as_float(sr[c0 + 2 * c]), __uint_as_float(sr[c0 + 2 * c + 1])), sl2x2, negm2);
      float x0, x1, p0, p1;
      unpack2(x, x0, x1);
      if ((pi % kEmuPeriod) < kEmuCount) {
        exp2_poly2(x0, x1, p0, p1);
      } else {
        p0 = (kDiag & 4) ? x0 * x0 : fast_exp2(x0);
        p1 = (kDiag & 4) ? x1 * x1 : fast_exp2(x1);
      }
      pr[c] = cvt_bf16x2(p0, p1);  // low half = key 2c, high half = key 2c+1
      if (c & 1) acc1 = add2(acc1, pack2(p0, p1));
      else acc0 = add2(acc0, pack2(p0, p1));
    }
    tmem_st16(s_addr + (uint32_t)(c0 / 2), pr);  // P overlays S (already in registers)
    if (c0 == 32) {
      // keys 0..63 of P are in TMEM: their P V starts while the second half is still being exponentiated,
      // which takes half a P V off the softmax -> P V -> Q K^T -> softmax latency chain of this tile
      tmem_wait_st();
      tc_fence_before();
      arrive_a();
      HGA_TR(3);
    }
  }
  float a0, a1;
  unpack2(add2(acc0, acc1), a0, a1);
  l_run += a0 + a1;
  tmem_wait_st();
  tc_fence_before();
  arrive_b();
  HGA_TR(4);
#undef HGA_TR
}

}  // namespace tc
}  // namespace hga
