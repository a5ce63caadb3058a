// peaks.cu - micro-benchmark behind the ALU roofline denominator: FADD / FADD2 / IADD / FHADD lane-adds per clock per SM and LDS.128 bytes per clock per SM.
// Build + run: nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o /tmp/peaks paper_1111_6399_b200/microbench/peaks.cu && /tmp/peaks
#include <cstdio>
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n",cudaGetErrorString(e),__LINE__);return 1;}}while(0)

template<int MODE> __global__ void __launch_bounds__(256) k_add(float *out, int iters, float seed) {
    float a[32];
    #pragma unroll
    for (int i=0;i<32;++i) a[i]=seed*i+threadIdx.x;
    float w0=seed, w1=seed*2;
    unsigned long long wp; asm("mov.b64 %0, {%1,%2};" : "=l"(wp) : "f"(w0), "f"(w1));
    for (int it=0; it<iters; ++it) {
        if (MODE==0) {
            #pragma unroll
            for (int r=0;r<4;++r)
            #pragma unroll
            for (int i=0;i<32;++i) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(a[i]) : "f"(w0));
        } else if (MODE==1) {
            #pragma unroll
            for (int r=0;r<4;++r)
            #pragma unroll
            for (int i=0;i<16;++i) {
                unsigned long long p; asm("mov.b64 %0, {%1,%2};" : "=l"(p) : "f"(a[2*i]), "f"(a[2*i+1]));
                asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(p) : "l"(wp));
                asm("mov.b64 {%0,%1}, %2;" : "=f"(a[2*i]), "=f"(a[2*i+1]) : "l"(p));
            }
        } else if (MODE==2) { // int add
            #pragma unroll
            for (int r=0;r<4;++r)
            #pragma unroll
            for (int i=0;i<32;++i) { int x=__float_as_int(a[i]); asm volatile("add.s32 %0, %0, %1;" : "+r"(x) : "r"(__float_as_int(w0))); a[i]=__int_as_float(x);}        
        } else if (MODE==3) { // mixed f32 += f16
            unsigned short h = __half_as_ushort(__float2half(w0));
            #pragma unroll
            for (int r=0;r<4;++r)
            #pragma unroll
            for (int i=0;i<32;++i) asm volatile("add.rn.f32.f16 %0, %1, %0;" : "+f"(a[i]) : "h"(h));
        }
    }
    float s=0;
    #pragma unroll
    for (int i=0;i<32;++i) s+=a[i];
    out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}

// LDS.128 bandwidth: each thread loads NV float4 per iter, conflict-free (consecutive lanes consecutive 16B)
__global__ void __launch_bounds__(256) k_lds(float *out, int iters) {
    extern __shared__ float4 sm[];
    for (int i=threadIdx.x;i<2048;i+=256) sm[i]=make_float4(i,1,2,3);
    __syncthreads();
    float4 acc=make_float4(0,0,0,0);
    int idx=threadIdx.x;
    for (int it=0;it<iters;++it){
        #pragma unroll
        for (int m=0;m<8;++m){ float4 v=sm[(idx+m*256)&2047]; acc.x+=v.x; acc.y+=v.y; acc.z+=v.z; acc.w+=v.w; }
        idx=(idx+1)&2047;
    }
    out[blockIdx.x*blockDim.x+threadIdx.x]=acc.x+acc.y+acc.z+acc.w;
}

int main(){
    float *d; CK(cudaMalloc(&d, 148*8*256*4*4));
    cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    int dev=0; cudaDeviceProp pr; cudaGetDeviceProperties(&pr,dev);
    printf("SMs %d clock %d kHz\n", pr.multiProcessorCount, pr.clockRate);
    const int iters=20000;
    for (int occ : {1,2,4}) {
      for (int mode=0; mode<4; ++mode){
        float ms=0;
        for (int rep=0;rep<3;++rep){
            cudaEventRecord(e0);
            int grid=148*occ;
            if(mode==0) k_add<0><<<grid,256>>>(d,iters,1.0f);
            if(mode==1) k_add<1><<<grid,256>>>(d,iters,1.0f);
            if(mode==2) k_add<2><<<grid,256>>>(d,iters,1.0f);
            if(mode==3) k_add<3><<<grid,256>>>(d,iters,1.0f);
            cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms,e0,e1);
        }
        double adds=(double)148*occ*256*iters*128;
        printf("mode %d (0 FADD,1 FADD2,2 IADD,3 FHADD) ctas/SM %d: %.3f ms  %.1f Gadds/s  = %.1f lane-adds/clk/SM @1965MHz\n", mode, occ, ms, adds/ms/1e6, adds/ms/1e6/148/1.965);
      }
    }
    for (int occ : {1,2,4}) {
        float ms=0;
        CK(cudaFuncSetAttribute(k_lds, cudaFuncAttributeMaxDynamicSharedMemorySize, 32768));
        for (int rep=0;rep<3;++rep){
            cudaEventRecord(e0);
            k_lds<<<148*occ,256,32768>>>(d,iters);
            cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms,e0,e1);
        }
        double bytes=(double)148*occ*256*iters*8*16;
        printf("LDS.128 ctas/SM %d: %.3f ms  %.1f B/clk/SM @1965MHz\n", occ, ms, bytes/ms/1e6/148/1.965);
    }
    return 0;
}
