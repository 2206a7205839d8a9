// microbenchmark (evidence for DESIGN.md section 7): the softmax tile of attend_tc2 (TMEM ld/st + hand-off) with the tensor pipe idle and
// while another warp of the same SM streams tcgen05 MMAs.  Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -I ../../../include -o t softmax_tile_with_mma.cu
#include <cstdio>
#include <cstdint>
#include <math_constants.h>
#include "../hga_attend_softmax.cuh"
using namespace hga::tc;
#define ITERS 256
template <int MODE, int EP, int EC, int TM>
__global__ void __launch_bounds__(384, 1) k(const float* in, float* out, long long* cyc, int nwarps, float sl2, int npoll) {
  const int warp = threadIdx.x / 32;
  __shared__ unsigned long long bar;
  __shared__ volatile int done;
  __shared__ uint32_t tmem_base_s;
  __shared__ unsigned long long bar2[16];
  if (threadIdx.x < 16) mbar_init(smem_u32(&bar2[threadIdx.x]), 1);
  if (threadIdx.x == 0) { mbar_init(smem_u32(&bar), 1); done = 0; }
  if (TM && warp == 0) tmem_alloc(smem_u32(&tmem_base_s), 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = TM ? tmem_base_s : 0u;
  const uint32_t s_addr = tmem + ((uint32_t)((warp % 4) * 32) << 16) + (uint32_t)((warp / 4) % 2) * 128u;
  if (warp == 8 && npoll == 9) {   // a tensor-pipe hog: M128 N128 K16 bf16 MMAs back to back until the softmax warps are done
    extern __shared__ __align__(1024) unsigned char dsm[];
    const uint32_t ld = elect_one();
    const uint32_t sb = smem_u32(dsm);
    constexpr uint32_t kDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);
    const uint32_t idesc = umma_idesc(128, 128, false);
    while (!done) {
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const uint32_t a = ((sb + (i % 4) * 32) & 0x3FFFFu) >> 4, b = ((sb + 32768 + (i % 4) * 32) & 0x3FFFFu) >> 4;
        umma_ss_e(tmem + 256, make_desc(a + (1u << 16), kDescHi), make_desc(b + (1u << 16), kDescHi), idesc, 1u, ld);
      }
      umma_commit_e(smem_u32(&bar2[15]), ld);
      __syncwarp();
    }
    // drain
    umma_commit_e(smem_u32(&bar2[14]), ld);
    mbar_wait(smem_u32(&bar2[14]), 0);
    return;
  }
  if (warp >= 8) {   // pollers
    if (warp - 8 < npoll) { while (!done) { if (mbar_try_wait(smem_u32(&bar), 0)) break; } }
    return;
  }
  uint32_t sr[128];
#pragma unroll
  for (int c = 0; c < 128; ++c) sr[c] = __float_as_uint(in[(threadIdx.x * 131 + c * 7) & 4095]);
  float m_run = 3.0f, l_run = 0.f;
  uint32_t keep = 0;
  asm volatile("bar.sync 1, 256;");
  long long t0 = clock64();
  if (warp < nwarps) {
    for (int it = 0; it < ITERS; ++it) {
      if (TM) {
        tmem_ld32(s_addr + 0, sr + 0); tmem_ld32(s_addr + 32, sr + 32); tmem_ld32(s_addr + 64, sr + 64); tmem_ld32(s_addr + 96, sr + 96);
        tmem_wait_ld();
      } else {
#pragma unroll
        for (int c = 0; c < 128; ++c) asm volatile("" : "+r"(sr[c]));  // opaque: fresh values each tile, no instruction
      }
      const uint64_t sl2x2 = pack2(sl2, sl2);
      if (MODE != 2) {
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
        if (__any_sync(0xffffffffu, (m_new - m_run) * sl2 > 8.f)) m_run = m_new;
      }
      if (MODE != 1) {
        const float neg_m = -m_run * sl2;
        const uint64_t negm2 = pack2(neg_m, neg_m);
        uint64_t acc0 = pack2(0.f, 0.f), acc1 = acc0;
#pragma unroll
        for (int c0 = 0; c0 < 128; c0 += 32) {
          uint32_t pr[16];
#pragma unroll
          for (int c = 0; c < 16; ++c) {
            const uint64_t x = fma2(pack2(__uint_as_float(sr[c0 + 2 * c]), __uint_as_float(sr[c0 + 2 * c + 1])), sl2x2, negm2);
            float x0, x1;
            unpack2(x, x0, x1);
            float p0, p1;
            if (((c0 / 2 + c) % EP) < EC) exp2_poly2(x0, x1, p0, p1);
            else { p0 = fast_exp2(x0); p1 = fast_exp2(x1); }
            pr[c] = cvt_bf16x2(p0, p1);
            if (c & 1) acc1 = add2(acc1, pack2(p0, p1)); else acc0 = add2(acc0, pack2(p0, p1));
          }
          if (TM) {
            tmem_st16(s_addr + (uint32_t)(c0 / 2), pr);
            if (TM == 2 && (c0 == 32 || c0 == 96)) { tmem_wait_st(); tc_fence_before(); __syncwarp(); if ((threadIdx.x & 31) == 0) mbar_arrive(smem_u32(&bar2[warp])); }
          } else {
#pragma unroll
            for (int c = 0; c < 16; ++c) keep ^= pr[c];
          }
        }
        float a0, a1;
        unpack2(add2(acc0, acc1), a0, a1);
        l_run += a0 + a1;
      }
    }
  }
  long long t1 = clock64();
  __syncwarp();
  if (warp < 8) { asm volatile("bar.sync 1, 256;"); if (threadIdx.x == 0) done = 1; }
  if (TM && warp == 0) { tc_fence_after(); tmem_dealloc(tmem, 512); }
  out[threadIdx.x] = l_run + m_run + (float)keep;
  if (threadIdx.x == 0) cyc[0] = t1 - t0;
}
int main() {
  float *in, *out; long long* cyc;
  cudaMalloc(&in, 4096 * 4); cudaMalloc(&out, 4096); cudaMalloc(&cyc, 8);
  float h[4096]; for (int i = 0; i < 4096; ++i) h[i] = (float)((i * 37) % 97) * 0.05f - 2.0f;
  cudaMemcpy(in, h, sizeof(h), cudaMemcpyHostToDevice);
  const char* names[] = {"max+exp (whole tile)", "max only", "exp only"};
  cudaFuncSetAttribute(k<0, 4, 0, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
  for (int v = 0; v < 2; ++v) for (int nw : {4, 8}) { int mode = 0; int npoll = v;
    if (v == 0) k<0, 4, 0, 2><<<1, 384, 65536>>>(in, out, cyc, nw, 0.1275f, 0);
    if (v == 1) k<0, 4, 0, 2><<<1, 384, 65536>>>(in, out, cyc, nw, 0.1275f, 9);
    cudaDeviceSynchronize(); long long c; cudaMemcpy(&c, cyc, 8, cudaMemcpyDeviceToHost);
    fflush(stdout); printf("variant %d (0: softmax tile with TMEM ld/st + hand-off, tensor pipe idle; 1: the same while another warp streams MMAs)  %-22s warps/scheduler %d: %.0f cycles per tile per warp (scheduler total per tile-set %.0f)\n", npoll, names[mode], nw / 4, (double)c / ITERS, (double)c / ITERS);
  }
  printf("%s\n", cudaGetErrorString(cudaGetLastError()));
}
