// tmem_cp.cu - B200 micro-benchmark behind DESIGN.md section 6 "why not tensor memory" (results: profiles/r2_microbench.md).
// Build + run: nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o /tmp/tmem_cp paper_1111_6399_b200/microbench/tmem_cp.cu && /tmp/tmem_cp
// tcgen05.cp probe: mapping of smem (matrix descriptor) -> TMEM lanes/columns, and throughput
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
__device__ __forceinline__ uint64_t mkdesc(unsigned saddr, unsigned lbo, unsigned sbo, unsigned layout){
  uint64_t d=0;
  d |= (uint64_t)((saddr>>4)&0x3fff);
  d |= (uint64_t)((lbo>>4)&0x3fff)<<16;
  d |= (uint64_t)((sbo>>4)&0x3fff)<<32;
  d |= (uint64_t)1<<46;
  d |= (uint64_t)layout<<61;
  return d;
}
#define LD8(r, base) asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n" \
 : "=r"(r[0]),"=r"(r[1]),"=r"(r[2]),"=r"(r[3]),"=r"(r[4]),"=r"(r[5]),"=r"(r[6]),"=r"(r[7]) : "r"(base))
__global__ void __launch_bounds__(128,1) kmap(unsigned layout, unsigned lbo, unsigned sbo, unsigned startoff, unsigned* out){
  extern __shared__ __align__(1024) unsigned char smem[];
  __shared__ unsigned taddr_s; __shared__ __align__(8) unsigned long long bar;
  unsigned* sw = (unsigned*)smem;
  for (int i=threadIdx.x;i<16384;i+=128) sw[i]=i;       // word index as value (64 KB)
  const int warp=threadIdx.x>>5;
  if (warp==0){
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 64;\n" :: "r"((unsigned)__cvta_generic_to_shared(&taddr_s)));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
  }
  if (threadIdx.x==0) asm volatile("mbarrier.init.shared.b64 [%0], 1;\n" :: "r"((unsigned)__cvta_generic_to_shared(&bar)));
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;\n");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n");
  const unsigned taddr=taddr_s;
  if (threadIdx.x==0){
    uint64_t d = mkdesc((unsigned)__cvta_generic_to_shared(smem)+startoff, lbo, sbo, layout);
    asm volatile("tcgen05.cp.cta_group::1.128x256b [%0], %1;\n" :: "r"(taddr), "l"(d) : "memory");
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" :: "r"((unsigned)__cvta_generic_to_shared(&bar)) : "memory");
  }
  asm volatile("{\n.reg .pred p;\nW: mbarrier.try_wait.parity.shared.b64 p, [%0], 0;\n@p bra D;\nbra W;\nD:\n}\n" :: "r"((unsigned)__cvta_generic_to_shared(&bar)) : "memory");
  asm volatile("tcgen05.fence::after_thread_sync;\n");
  unsigned r[8];
  LD8(r, taddr + ((32u*warp)<<16));
  asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
  for(int k=0;k<8;k++) out[threadIdx.x*8+k]=r[k];
  __syncthreads();
  if (warp==0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 64;\n" :: "r"(taddr));
}
__global__ void __launch_bounds__(128,1) kbw(int iters, int ncp, long long* cyc){
  extern __shared__ __align__(1024) unsigned char smem[];
  __shared__ unsigned taddr_s; __shared__ __align__(8) unsigned long long bar;
  const int warp=threadIdx.x>>5;
  if (warp==0){
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;\n" :: "r"((unsigned)__cvta_generic_to_shared(&taddr_s)));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
  }
  if (threadIdx.x==0) asm volatile("mbarrier.init.shared.b64 [%0], 1;\n" :: "r"((unsigned)__cvta_generic_to_shared(&bar)));
  asm volatile("tcgen05.fence::before_thread_sync;\n");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n");
  const unsigned taddr=taddr_s;
  if (threadIdx.x==0){
    long long t0=clock64();
    unsigned par=0;
    for(int it=0;it<iters;it++){
      for(int j=0;j<ncp;j++){
        uint64_t d = mkdesc((unsigned)__cvta_generic_to_shared(smem)+ (j&7)*4096, 128, 256, 0);
        asm volatile("tcgen05.cp.cta_group::1.128x256b [%0], %1;\n" :: "r"(taddr+ (j*8)%512), "l"(d) : "memory");
      }
      asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" :: "r"((unsigned)__cvta_generic_to_shared(&bar)) : "memory");
      asm volatile("{\n.reg .pred p;\nW2: mbarrier.try_wait.parity.shared.b64 p, [%0], %1;\n@p bra D2;\nbra W2;\nD2:\n}\n" :: "r"((unsigned)__cvta_generic_to_shared(&bar)), "r"(par) : "memory");
      par^=1;
    }
    long long t1=clock64();
    cyc[blockIdx.x]=t1-t0;
  }
  __syncthreads();
  if (warp==0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;\n" :: "r"(taddr));
}
int main(){
  unsigned* out; cudaMalloc(&out,128*8*4); unsigned h[1024];
  cudaFuncSetAttribute(kmap, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
  cudaFuncSetAttribute(kbw, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
  struct T{unsigned layout,lbo,sbo,off; const char* name;} tests[]={
    {0,128,256,0,"noswz lbo128 sbo256"},
    {0,2048,128,0,"noswz lbo2048 sbo128"},
    {2,16,1024,0,"sw128 sbo1024"},
    {2,16,1024,32,"sw128 sbo1024 +32B"},
    {2,16,1024,128,"sw128 sbo1024 +128B"},
    {4,16,512,0,"sw64 sbo512"},
    {4,16,512,32,"sw64 sbo512 +32B"},
    {4,16,512,64,"sw64 sbo512 +64B"},
    {6,16,256,0,"sw32 sbo256"},
  };
  for (auto&t: tests){
    cudaMemset(out,0xff,4096);
    kmap<<<1,128,65536>>>(t.layout,t.lbo,t.sbo,t.off,out); cudaError_t e=cudaDeviceSynchronize();
    cudaMemcpy(h,out,4096,cudaMemcpyDeviceToHost);
    printf("%s: %s\n",t.name,cudaGetErrorString(e));
    for(int lane: {0,1,2,7,8,9,31,32,127}){ printf("  lane %3d:",lane); for(int k=0;k<8;k++) printf(" %5u",h[lane*8+k]); printf("\n"); }
  }
  long long* cyc; cudaMalloc(&cyc,148*8); long long hc[148];
  for(int ncp: {1,4,16,64}){
    kbw<<<148,128,65536>>>(200,ncp,cyc); cudaError_t e=cudaDeviceSynchronize();
    cudaMemcpy(hc,cyc,148*8,cudaMemcpyDeviceToHost);
    printf("cp 128x256b x%d per commit: %s %lld cycles -> %.1f B/clk/SM\n",ncp,cudaGetErrorString(e),hc[0],200.0*ncp*4096/hc[0]);
  }
  return 0;
}
