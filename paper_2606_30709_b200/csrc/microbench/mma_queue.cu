// microbenchmark (evidence for DESIGN.md section 7): how deep is the tcgen05.mma issue queue?  One thread issues 24 MMAs
// (M128 N128 K16, bf16, SS or TS) back to back and timestamps every issue; then commit + wait.
// Build and run on a B200 (from this directory):
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -I ../../../include -o mma_queue mma_queue.cu && ./mma_queue
#include <cstdio>
#include <cstdint>
#include "../hga_tc_ptx.cuh"
using namespace hga::tc;
template <int TS>
__global__ void __launch_bounds__(128, 1) k(long long* out) {
  extern __shared__ __align__(1024) unsigned char smem[];
  __shared__ unsigned long long bar;
  __shared__ uint32_t tbase;
  const int warp = threadIdx.x / 32;
  for (int i = threadIdx.x; i < 65536 / 4; i += 128) reinterpret_cast<uint32_t*>(smem)[i] = 0x3c003c00u;
  if (threadIdx.x == 0) { mbar_init(smem_u32(&bar), 1); fence_barrier_init(); }
  if (warp == 0) tmem_alloc(smem_u32(&tbase), 512);
  fence_proxy_async();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tbase;
  if (warp == 1) {
    const uint32_t ld = elect_one();
    const uint32_t sb = smem_u32(smem);
    constexpr uint32_t kDescHi = (1024u >> 4) | (1u << 14) | (2u << 29);
    const uint32_t idesc = umma_idesc(128, 128, false);
    const uint32_t idesc_pv = umma_idesc(128, 128, true);
    long long ts[26];
    ts[0] = clock64();
#pragma unroll
    for (int i = 0; i < 24; ++i) {
      const uint32_t a = ((sb + (i % 4) * 32) & 0x3FFFFu) >> 4, b = ((sb + 32768 + (i % 4) * 32) & 0x3FFFFu) >> 4;
      if (TS) umma_ts_e(tmem + 256, tmem + (uint32_t)((i % 8) * 8), make_desc(b + ((16384u >> 4) << 16), kDescHi), idesc_pv, 1u, ld);
      else umma_ss_e(tmem + (uint32_t)((i / 8 % 2) * 128), make_desc(a + (1u << 16), kDescHi), make_desc(b + (1u << 16), kDescHi), idesc, (i % 8) ? 1u : 0u, ld);
      ts[i + 1] = clock64();
    }
    umma_commit_e(smem_u32(&bar), ld);
    mbar_wait(smem_u32(&bar), 0);
    ts[25] = clock64();
    if (ld) for (int i = 0; i < 26; ++i) out[i] = ts[i] - ts[0];
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) { tc_fence_after(); tmem_dealloc(tmem, 512); }
}
int main() {
  long long* out; cudaMalloc(&out, 26 * 8);
  for (int ts = 0; ts < 2; ++ts) {
    if (ts) { cudaFuncSetAttribute(k<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536); k<1><<<1, 128, 65536>>>(out); }
    else { cudaFuncSetAttribute(k<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536); k<0><<<1, 128, 65536>>>(out); }
    cudaDeviceSynchronize();
    long long h[26]; cudaMemcpy(h, out, sizeof(h), cudaMemcpyDeviceToHost);
    printf("%s: issue timestamps (cycles after the first):", ts ? "TS (A in TMEM)" : "SS");
    for (int i = 1; i <= 24; ++i) printf(" %lld", h[i]);
    printf(" | all complete at %lld  (%s)\n", h[25], cudaGetErrorString(cudaGetLastError()));
  }
}
