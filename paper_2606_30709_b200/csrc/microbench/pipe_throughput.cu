// microbenchmark (evidence for DESIGN.md section 7): per-scheduler throughput of MUFU.EX2 f32 / f16x2 / bf16x2, FFMA2, FMNMX3, FFMA.
// Build and run on a B200:  nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o pipe_throughput pipe_throughput.cu && ./pipe_throughput
#include <cstdio>
#include <cstdint>
#include <cuda_fp16.h>
#include <cuda_bf16.h>
#define ITERS 4096
__device__ __forceinline__ float ex2f(float x){float y; asm volatile("ex2.approx.ftz.f32 %0, %1;":"=f"(y):"f"(x)); return y;}
__device__ __forceinline__ uint32_t ex2h2(uint32_t x){uint32_t y; asm volatile("ex2.approx.f16x2 %0, %1;":"=r"(y):"r"(x)); return y;}
__device__ __forceinline__ uint32_t ex2b2(uint32_t x){uint32_t y; asm volatile("ex2.approx.ftz.bf16x2 %0, %1;":"=r"(y):"r"(x)); return y;}
__device__ __forceinline__ uint64_t fma2(uint64_t a,uint64_t b,uint64_t c){uint64_t r; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;":"=l"(r):"l"(a),"l"(b),"l"(c)); return r;}
template<int MODE> __global__ void k(float* out, long long* cyc, int nwarps_active){
  int warp = threadIdx.x/32;
  float a[8]; uint32_t u[8]; uint64_t w[8];
  for(int i=0;i<8;i++){a[i]=-0.001f*(threadIdx.x+i); u[i]=0xb800b800u+i+threadIdx.x; w[i]=((uint64_t)__float_as_uint(0.5f+i)<<32)|__float_as_uint(0.25f+threadIdx.x);}
  __syncthreads();
  long long t0=clock64();
  if (warp < nwarps_active) {
  for(int it=0;it<ITERS;it++){
    #pragma unroll
    for(int i=0;i<8;i++){
      if(MODE==0) a[i]=ex2f(a[i]);
      if(MODE==1) u[i]=ex2h2(u[i]);
      if(MODE==2) u[i]=ex2b2(u[i]);
      if(MODE==3) w[i]=fma2(w[i],w[i],w[i]);
      if(MODE==4) { asm volatile("max.f32 %0, %0, %1, %2;":"+f"(a[i]):"f"(a[(i+1)&7]),"f"(a[(i+2)&7])); }
      if(MODE==5) { asm volatile("cvt.rn.bf16x2.f32 %0, %1, %2;":"=r"(u[i]):"f"(a[i]),"f"(a[(i+1)&7])); }
      if(MODE==6) { asm volatile("shf.l.wrap.b32 %0, %1, %1, 23;":"=r"(u[i]):"r"(u[i])); asm volatile("add.u32 %0, %0, %1;":"+r"(u[i]):"r"(u[(i+1)&7])); }
      if(MODE==7) { a[i]=ex2f(a[i]); w[i]=fma2(w[i],w[i],w[i]); }   // mixed: 1 MUFU + 1 FFMA2
      if(MODE==8) { a[i]=ex2f(a[i]); w[i]=fma2(w[i],w[i],w[i]); w[(i+4)&7]=fma2(w[(i+4)&7],w[i],w[i]); w[(i+2)&7]=fma2(w[(i+2)&7],w[i],w[i]);}   // 1 MUFU + 3 FFMA2
      if(MODE==9) { asm volatile("fma.rn.f32 %0, %0, %0, %0;":"+f"(a[i])); }
    }
  }
  }
  long long t1=clock64();
  float s=0; for(int i=0;i<8;i++) s+=a[i]+u[i]+(float)w[i];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
  if(threadIdx.x==0) cyc[blockIdx.x]=t1-t0;
}
int main(){
  float* out; long long* cyc; cudaMalloc(&out, 148*1024*4); cudaMalloc(&cyc, 148*8);
  const char* names[]={"ex2.f32","ex2.f16x2","ex2.bf16x2","fma.f32x2","max3.f32","cvt.bf16x2","shl+add","ex2+fma2","ex2+3fma2","ffma"};
  for(int mode=0;mode<10;mode++) for(int nw: {4,8,16}){
    #define L(M) case M: k<M><<<1,512>>>(out,cyc,nw); break;
    switch(mode){L(0)L(1)L(2)L(3)L(4)L(5)L(6)L(7)L(8)L(9)}
    cudaDeviceSynchronize(); long long c; cudaMemcpy(&c,cyc,8,cudaMemcpyDeviceToHost);
    // per SMSP: nw/4 warps, each ITERS*8 ops
    double per = (double)c/(ITERS*8.0*(nw/4));
    printf("%-12s warps/SMSP=%d  cycles per warp-instr(group) per SMSP = %.2f\n", names[mode], nw/4, per);
  }
  printf("%s\n", cudaGetErrorString(cudaGetLastError()));
}
