// microbenchmark (evidence for DESIGN.md section 7): dependent-chain latency of the softmax instruction mix (one warp, one chain).
// Build and run on a B200:  nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o pipe_latency pipe_latency.cu && ./pipe_latency
#include <cstdio>
#include <cstdint>
#define ITERS 2048
template<int MODE> __global__ void k(float* out, long long* cyc){
  float a=threadIdx.x*0.001f, b=1.0001f, c=0.5f; uint64_t w=((uint64_t)__float_as_uint(0.5f)<<32)|__float_as_uint(0.25f+threadIdx.x); uint32_t u=threadIdx.x;
  long long t0=clock64();
  #pragma unroll 16
  for(int it=0;it<ITERS;it++){
    if(MODE==0) asm volatile("max.f32 %0, %0, %1, %2;":"+f"(a):"f"(b),"f"(c));
    if(MODE==1) asm volatile("max.f32 %0, %0, %1;":"+f"(a):"f"(b));
    if(MODE==2) asm volatile("fma.rn.f32x2 %0, %0, %0, %0;":"+l"(w));
    if(MODE==3) asm volatile("add.rn.f32x2 %0, %0, %0;":"+l"(w));
    if(MODE==4) asm volatile("ex2.approx.ftz.f32 %0, %0;":"+f"(a));
    if(MODE==5) { asm volatile("cvt.rn.bf16x2.f32 %0, %1, %1;":"=r"(u):"f"(a)); a=__uint_as_float(u); }
    if(MODE==6) asm volatile("fma.rn.f32 %0, %0, %0, %0;":"+f"(a));
    if(MODE==7) { asm volatile("shl.b32 %0, %0, 23;":"+r"(u)); asm volatile("add.u32 %0, %0, %0;":"+r"(u)); }
  }
  long long t1=clock64();
  out[threadIdx.x]=a+(float)w+u;
  if(threadIdx.x==0) cyc[0]=t1-t0;
}
int main(){
  float* out; long long* cyc; cudaMalloc(&out, 4096); cudaMalloc(&cyc, 8);
  const char* names[]={"max3","max2","fma2","add2","ex2","cvt.bf16x2","ffma","shl+add"};
  for(int mode=0;mode<8;mode++){
    #define L(M) case M: k<M><<<1,32>>>(out,cyc); break;
    switch(mode){L(0)L(1)L(2)L(3)L(4)L(5)L(6)L(7)}
    cudaDeviceSynchronize(); long long c; cudaMemcpy(&c,cyc,8,cudaMemcpyDeviceToHost);
    printf("%-10s latency %.2f cycles\n", names[mode], (double)c/ITERS);
  }
  printf("%s\n", cudaGetErrorString(cudaGetLastError()));
}
