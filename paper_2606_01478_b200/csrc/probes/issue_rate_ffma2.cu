// issue_rate_ffma2.cu -- standalone micro-benchmark (not part of libcf.so): FP32 FMA issue rate on B200, packed FFMA2
// (fma.rn.f32x2) vs scalar FFMA, alone and mixed with ALU-pipe LOP3.  Result: profiles/r1_microbench_ffma2.md.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/issue_rate_ffma2 paper_2606_01478_b200/csrc/probes/issue_rate_ffma2.cu
#include <cstdio>
#include <cuda_runtime.h>
typedef unsigned long long u64;
__device__ __forceinline__ u64 pk(float a, float b){ u64 r; asm("mov.b64 %0, {%1,%2};":"=l"(r):"f"(a),"f"(b)); return r;}
__device__ __forceinline__ void upk(u64 r, float&a, float&b){ asm("mov.b64 {%0,%1}, %2;":"=f"(a),"=f"(b):"l"(r));}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c){ u64 r; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;":"=l"(r):"l"(a),"l"(b),"l"(c)); return r;}
__device__ __forceinline__ float fma1(float a, float b, float c){ float r; asm volatile("fma.rn.f32 %0, %1, %2, %3;":"=f"(r):"f"(a),"f"(b),"f"(c)); return r;}
__device__ __forceinline__ unsigned lop(unsigned a, unsigned b){ unsigned r; asm volatile("xor.b32 %0, %1, %2;":"=r"(r):"r"(a),"r"(b)); return r;}
// MODE 0: 16 FFMA ; 1: 8 FFMA2 ; 2: 16 FFMA + 16 LOP ; 3: 8 FFMA2 + 16 LOP ; 4: 16 LOP
template<int MODE> __global__ void k(float* out, int iters, float s){
  float a[16]; u64 p[8]; unsigned z[16];
  for (int j=0;j<16;++j){ a[j]=threadIdx.x*0.001f+j; z[j]=threadIdx.x+j; }
  for (int j=0;j<8;++j) p[j]=pk(a[2*j],a[2*j+1]);
  u64 S=pk(s,s), C=pk(0.5f,0.25f);
  for (int t=0;t<iters;++t){
    if (MODE==0||MODE==2){
      #pragma unroll
      for (int j=0;j<16;++j) a[j]=fma1(a[j],s,0.5f);
    }
    if (MODE==1||MODE==3){
      #pragma unroll
      for (int j=0;j<8;++j) p[j]=fma2(p[j],S,C);
    }
    if (MODE>=2){
      #pragma unroll
      for (int j=0;j<16;++j) z[j]=lop(z[j],z[(j+1)&15]);
    }
  }
  float r=0; unsigned zz=0;
  for (int j=0;j<16;++j){ r+=a[j]; zz^=z[j]; }
  for (int j=0;j<8;++j){ float x,y; upk(p[j],x,y); r+=x+y; }
  out[blockIdx.x*blockDim.x+threadIdx.x]=r+zz;
}
template<int MODE> void run(const char* name, float* out){
  int iters=20000; dim3 g(148*8), b(256);
  k<MODE><<<g,b>>>(out,10,1.0001f); cudaDeviceSynchronize();
  cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  cudaEventRecord(e0); k<MODE><<<g,b>>>(out,iters,1.0001f); cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms,e0,e1);
  double warps=148.0*8*8, winst_fp = (MODE==4?0:16.0)*iters*warps; // FFMA-equivalent warp-instrs
  double cyc = ms*1e-3*1.965e9; // assume max clock
  printf("%-28s %8.3f ms  FMA-equiv warp-inst/clk/SM = %.2f  (lane-fma/clk/SM = %.1f)\n", name, ms, winst_fp/cyc/148, 32*winst_fp/cyc/148);
}
int main(){ float* out; cudaMalloc(&out, 148*8*256*4);
  run<0>("16 FFMA",out); run<1>("8 FFMA2",out); run<2>("16 FFMA + 16 LOP",out); run<3>("8 FFMA2 + 16 LOP",out); run<4>("16 LOP",out);
  return 0; }
