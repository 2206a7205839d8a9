// microbenchmark (evidence for DESIGN.md section 7, S2): per-scheduler throughput of DFMA and of the fp64 tensor-core
// instruction mma.sync.m8n8k4.f64 on one SM, 1 / 2 / 4 warps per scheduler.
// Build and run on a B200:  nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o fp64_throughput fp64_throughput.cu && ./fp64_throughput
#include <cstdio>
#include <cstdint>
#define ITERS 2048
template <int MODE>
__global__ void k(double* out, long long* cyc, int nwarps_active) {
  const int warp = threadIdx.x / 32;
  double a[8], c0[8], c1[8];
  for (int i = 0; i < 8; i++) { a[i] = 1.0 + 1e-9 * (threadIdx.x + i); c0[i] = 0.5 * i; c1[i] = 0.25 * i; }
  __syncthreads();
  const long long t0 = clock64();
  if (warp < nwarps_active) {
    for (int it = 0; it < ITERS; it++) {
#pragma unroll
      for (int i = 0; i < 8; i++) {
        if (MODE == 0) asm volatile("fma.rn.f64 %0, %1, %1, %0;" : "+d"(c0[i]) : "d"(a[i]));
        if (MODE == 1)  // D (8x8) = A (8x4) * B (4x8) + C: 256 FMAs per warp instruction
          asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                       : "+d"(c0[i]), "+d"(c1[i]) : "d"(a[i]), "d"(a[(i + 1) & 7]));
      }
    }
  }
  const long long t1 = clock64();
  double s = 0;
  for (int i = 0; i < 8; i++) s += c0[i] + c1[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
  if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}
int main() {
  double* out; long long* cyc;
  cudaMalloc(&out, 1024 * 8); cudaMalloc(&cyc, 8);
  const char* names[] = {"DFMA (32 FMA per warp instr)", "DMMA m8n8k4 (256 FMA per warp instr)"};
  for (int mode = 0; mode < 2; mode++)
    for (int nw : {4, 8, 16}) {
      if (mode == 0) k<0><<<1, 512>>>(out, cyc, nw); else k<1><<<1, 512>>>(out, cyc, nw);
      cudaDeviceSynchronize();
      long long c; cudaMemcpy(&c, cyc, 8, cudaMemcpyDeviceToHost);
      const double per = (double)c / (ITERS * 8.0 * (nw / 4));
      const double fma_per_clk_sm = (mode == 0 ? 32.0 : 256.0) / per * 4.0;
      printf("%-38s warps/SMSP=%d  cycles per warp instr per SMSP = %.2f  -> %.1f FMA/clk/SM\n", names[mode], nw / 4, per, fma_per_clk_sm);
    }
  printf("%s\n", cudaGetErrorString(cudaGetLastError()));
}
