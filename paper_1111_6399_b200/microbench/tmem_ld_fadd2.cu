// tmem_ld_fadd2.cu - B200 micro-benchmark behind DESIGN.md section 6 "why not tensor memory" (results: profiles/r2_microbench.md).
// Build + run: nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o /tmp/tmem_ld_fadd2 paper_1111_6399_b200/microbench/tmem_ld_fadd2.cu && /tmp/tmem_ld_fadd2
// how do LDTM.x16 and FADD2 share the SMSP? per iteration: NL x (LDTM.x16) and NF FADD2 on independent accumulators
#include <cstdio>
#include <cuda_runtime.h>
typedef unsigned long long u64;
#define LD16(r, base) asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n" \
 : "=r"(r[0]),"=r"(r[1]),"=r"(r[2]),"=r"(r[3]),"=r"(r[4]),"=r"(r[5]),"=r"(r[6]),"=r"(r[7]),"=r"(r[8]),"=r"(r[9]),"=r"(r[10]),"=r"(r[11]),"=r"(r[12]),"=r"(r[13]),"=r"(r[14]),"=r"(r[15]) : "r"(base))
template<int NL,int NF>
__global__ void __launch_bounds__(512,1) k(int iters, float* out, long long* cyc){
  __shared__ unsigned taddr_s;
  const int warp = threadIdx.x>>5;
  if (warp==0){
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;\n" :: "r"((unsigned)__cvta_generic_to_shared(&taddr_s)));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n");
  const unsigned taddr = taddr_s + ((32u*(warp&3))<<16);
  u64 acc[16]; for(int i=0;i<16;i++) acc[i]=0;
  u64 one = 0x3f8000003f800000ull;
  unsigned r[16]; unsigned x=0;
  long long t0=clock64();
  for(int it=0;it<iters;it++){
    #pragma unroll
    for(int l=0;l<NL;l++){ LD16(r, taddr + ((it*5+l*16)&255)); asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory"); x^=r[0]^r[15]; }
    #pragma unroll
    for(int f=0;f<NF;f++) asm volatile("add.rn.f32x2 %0, %0, %1;\n" : "+l"(acc[f&15]) : "l"(one));
  }
  long long t1=clock64();
  float s=0; for(int i=0;i<16;i++) s+=__uint_as_float((unsigned)acc[i]);
  out[blockIdx.x*blockDim.x+threadIdx.x]=s+x;
  if(threadIdx.x==0) cyc[blockIdx.x]=t1-t0;
  __syncthreads();
  if (warp==0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;\n" :: "r"(taddr_s));
}
template<int NL,int NF> void run(float* out,long long* cyc,int threads){
  long long hc[148]; int iters=4000;
  for(int rep=0;rep<2;rep++){ k<NL,NF><<<148,threads>>>(iters,out,cyc); cudaDeviceSynchronize(); }
  cudaMemcpy(hc,cyc,148*8,cudaMemcpyDeviceToHost);
  double per_smsp = (double)hc[0]/iters/(threads/128.0);   // cycles per iteration per warp-slot on an SMSP
  printf("threads %d NL=%d NF=%d: %.1f cyc/iter/warp -> per SMSP per iter %.1f cyc (LDTM alone would be %d x ?, FADD2 alone %d)\n",threads,NL,NF,(double)hc[0]/iters,per_smsp,NL,NF*2);
}
int main(){
  float* out; long long* cyc; cudaMalloc(&out,148*512*4); cudaMalloc(&cyc,148*8);
  for(int threads: {128,512}){
    run<1,0>(out,cyc,threads); run<0,8>(out,cyc,threads); run<1,8>(out,cyc,threads); run<1,16>(out,cyc,threads); run<1,32>(out,cyc,threads); run<2,8>(out,cyc,threads); run<4,8>(out,cyc,threads);
  }
  return 0;
}
