// branch_cost.cu - warp latency of an indirect branch (brx.idx -> LDC + BRX) vs a 3-level tree of direct predicated branches (SUBBAND dispatch).
// Build + run: nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o /tmp/branch_cost paper_1111_6399_b200/microbench/branch_cost.cu && /tmp/branch_cost
#include <cstdio>
#include <cuda_runtime.h>
__global__ void k_brx(unsigned* out, int n, unsigned seed, long long* cyc){
  unsigned x=seed ^ out[32+(threadIdx.x&0)], acc=0;
  long long t0=clock64();
  #pragma unroll 1
  for(int i=0;i<n;++i){
    asm volatile("{\n .reg .b32 t;\n and.b32 t, %1, 7;\n"
      "TB: .branchtargets B0,B1,B2,B3,B4,B5,B6,B7;\n brx.idx.uni t, TB;\n"
      "B0: add.u32 %0, %0, 1; bra.uni E;\n B1: add.u32 %0, %0, 3; bra.uni E;\n B2: add.u32 %0, %0, 5; bra.uni E;\n B3: add.u32 %0, %0, 7; bra.uni E;\n"
      "B4: add.u32 %0, %0, 9; bra.uni E;\n B5: add.u32 %0, %0, 11; bra.uni E;\n B6: add.u32 %0, %0, 13; bra.uni E;\n B7: add.u32 %0, %0, 15; bra.uni E;\n E:\n}"
      : "+r"(acc) : "r"(x));
    x = x*1664525u+1013904223u; x = (x>>13)^x;
  }
  long long t1=clock64();
  out[threadIdx.x]=acc+x; if(threadIdx.x==0) cyc[0]=t1-t0;
}
__global__ void k_tree(unsigned* out, int n, unsigned seed, long long* cyc){
  unsigned x=seed ^ out[32+(threadIdx.x&0)], acc=0;
  long long t0=clock64();
  #pragma unroll 1
  for(int i=0;i<n;++i){
    asm volatile("{\n .reg .pred p0,p1,p2;\n .reg .b32 t;\n and.b32 t, %1, 1; setp.ne.u32 p0, t, 0; and.b32 t, %1, 2; setp.ne.u32 p1, t, 0; and.b32 t, %1, 4; setp.ne.u32 p2, t, 0;\n"
      "@p2 bra.uni H; @p1 bra.uni L1; @p0 bra.uni B1; add.u32 %0,%0,1; bra.uni E; B1: add.u32 %0,%0,3; bra.uni E;\n"
      "L1: @p0 bra.uni B3; add.u32 %0,%0,5; bra.uni E; B3: add.u32 %0,%0,7; bra.uni E;\n"
      "H: @p1 bra.uni H1; @p0 bra.uni B5; add.u32 %0,%0,9; bra.uni E; B5: add.u32 %0,%0,11; bra.uni E;\n"
      "H1: @p0 bra.uni B7; add.u32 %0,%0,13; bra.uni E; B7: add.u32 %0,%0,15; bra.uni E;\n E:\n}"
      : "+r"(acc) : "r"(x));
    x = x*1664525u+1013904223u; x = (x>>13)^x;
  }
  long long t1=clock64();
  out[threadIdx.x]=acc+x; if(threadIdx.x==0) cyc[0]=t1-t0;
}
__global__ void k_none(unsigned* out, int n, unsigned seed, long long* cyc){
  unsigned x=seed ^ out[32+(threadIdx.x&0)], acc=0;
  long long t0=clock64();
  #pragma unroll 1
  for(int i=0;i<n;++i){
    asm volatile("add.u32 %0, %0, %1;" : "+r"(acc) : "r"(x&7));
    x = x*1664525u+1013904223u; x = (x>>13)^x;
  }
  long long t1=clock64();
  out[threadIdx.x]=acc+x; if(threadIdx.x==0) cyc[0]=t1-t0;
}
int main(){
  unsigned* o; long long* c; cudaMalloc(&o,4096); cudaMallocManaged(&c,8);
  int n=100000;
  for(int w: {1,2,4,8}){
    k_none<<<1,32*w>>>(o,n,12345,c); cudaDeviceSynchronize(); double a=(double)c[0]/n;
    k_brx<<<1,32*w>>>(o,n,12345,c); cudaDeviceSynchronize(); double b=(double)c[0]/n;
    k_tree<<<1,32*w>>>(o,n,12345,c); cudaDeviceSynchronize(); double t=(double)c[0]/n;
    printf("warps/CTA %d: loop-only %.1f cyc/iter, brx.idx %.1f, 3-level tree %.1f\n", w,a,b,t);
  }
  return 0;
}
