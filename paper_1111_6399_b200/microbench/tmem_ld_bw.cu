// tmem_ld_bw.cu - B200 micro-benchmark behind DESIGN.md section 6 "why not tensor memory" (results: profiles/r2_microbench.md).
// Build + run: nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o /tmp/tmem_ld_bw paper_1111_6399_b200/microbench/tmem_ld_bw.cu && /tmp/tmem_ld_bw
// tcgen05.ld throughput probe: bytes/clk/SM for 32x32b.x32 loads at arbitrary column offsets
#include <cstdio>
#include <cuda_runtime.h>
#define LD32(base) asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];\n" \
 : "=r"(r[0]),"=r"(r[1]),"=r"(r[2]),"=r"(r[3]),"=r"(r[4]),"=r"(r[5]),"=r"(r[6]),"=r"(r[7]),"=r"(r[8]),"=r"(r[9]),"=r"(r[10]),"=r"(r[11]),"=r"(r[12]),"=r"(r[13]),"=r"(r[14]),"=r"(r[15]),"=r"(r[16]),"=r"(r[17]),"=r"(r[18]),"=r"(r[19]),"=r"(r[20]),"=r"(r[21]),"=r"(r[22]),"=r"(r[23]),"=r"(r[24]),"=r"(r[25]),"=r"(r[26]),"=r"(r[27]),"=r"(r[28]),"=r"(r[29]),"=r"(r[30]),"=r"(r[31]) : "r"(base))
template<int MODE>
__global__ void __launch_bounds__(512) k(int iters, unsigned* out, long long* cyc){
  __shared__ unsigned taddr_s;
  const int warp = threadIdx.x>>5;
  if (warp==0){
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;\n" :: "r"((unsigned)__cvta_generic_to_shared(&taddr_s)));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n");
  unsigned taddr = taddr_s + ((32u*(warp&3))<<16);
  unsigned r[32], s[32]; unsigned acc=0;
  float fa[16]; for(int i=0;i<16;i++) fa[i]=threadIdx.x+i;
  long long t0=clock64();
  for(int i=0;i<iters;i++){
    unsigned col = (i*7)&127;
    LD32(taddr+col);
    if (MODE==1){
      #pragma unroll
      for(int q=0;q<16;q++) fa[q]+= __uint_as_float(acc)+1.0f;   // some FP work between
    }
    asm volatile("tcgen05.wait::ld.sync.aligned;\n");
    acc ^= r[0]^r[13]^r[31];
  }
  long long t1=clock64();
  float fs=0; for(int i=0;i<16;i++) fs+=fa[i];
  out[blockIdx.x*blockDim.x+threadIdx.x]=acc+(unsigned)fs;
  if(threadIdx.x==0) cyc[blockIdx.x]=t1-t0;
  __syncthreads();
  if (warp==0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;\n" :: "r"(taddr_s));
}
// two loads in flight
__global__ void __launch_bounds__(512) k2(int iters, unsigned* out, long long* cyc){
  __shared__ unsigned taddr_s;
  const int warp = threadIdx.x>>5;
  if (warp==0){
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;\n" :: "r"((unsigned)__cvta_generic_to_shared(&taddr_s)));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n");
  unsigned taddr = taddr_s + ((32u*(warp&3))<<16);
  unsigned acc=0;
  long long t0=clock64();
  for(int i=0;i<iters;i++){
    unsigned col = (i*7)&127;
    { unsigned r[32]; LD32(taddr+col); unsigned s2[32];
      { unsigned* r=s2; LD32(taddr+col+33); }
      asm volatile("tcgen05.wait::ld.sync.aligned;\n");
      acc ^= r[0]^r[13]^r[31]^s2[1]^s2[30]; }
  }
  long long t1=clock64();
  out[blockIdx.x*blockDim.x+threadIdx.x]=acc;
  if(threadIdx.x==0) cyc[blockIdx.x]=t1-t0;
  __syncthreads();
  if (warp==0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;\n" :: "r"(taddr_s));
}
int main(){
  unsigned* out; long long* cyc; cudaMalloc(&out, 148*512*4); cudaMalloc(&cyc,148*8);
  long long h[148];
  int iters=20000;
  for(int threads: {32,128,256,512}){
    k<0><<<148,threads>>>(iters,out,cyc); cudaDeviceSynchronize();
    k<0><<<148,threads>>>(iters,out,cyc); cudaError_t e=cudaDeviceSynchronize();
    cudaMemcpy(h,cyc,148*8,cudaMemcpyDeviceToHost);
    double bytes=(double)iters*32*4*threads;
    printf("x32 1-in-flight threads %d: %s cycles %lld  -> %.1f B/clk/SM (%.1f per warp-slot)\n",threads,cudaGetErrorString(e),h[0],bytes/h[0], bytes/h[0]/(threads/32));
    k2<<<148,threads>>>(iters,out,cyc); e=cudaDeviceSynchronize();
    cudaMemcpy(h,cyc,148*8,cudaMemcpyDeviceToHost);
    printf("x32 2-in-flight threads %d: %s cycles %lld  -> %.1f B/clk/SM\n",threads,cudaGetErrorString(e),h[0],2*bytes/h[0]);
    k<1><<<148,threads>>>(iters,out,cyc); e=cudaDeviceSynchronize();
    cudaMemcpy(h,cyc,148*8,cudaMemcpyDeviceToHost);
    printf("x32 + 16 FADD threads %d: %s cycles %lld  -> %.1f B/clk/SM\n",threads,cudaGetErrorString(e),h[0],bytes/h[0]);
  }
  return 0;
}
