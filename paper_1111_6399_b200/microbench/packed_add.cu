// packed_add.cu - can u8 data be summed faster as packed 16-bit pairs on the integer pipes than as fp32?
// One thread = 4 DM rows x 26 accumulator words + a 32-word window reloaded from shared memory every
// "channel" (16 LDS.64, lane stride 26 words: conflict-free), 12 warps per SM, like the SUBBAND consumers
// but with static offsets and no dispatch. Modes:
//   0  fp32, even offsets: 13 FADD2 per row and channel (26 samples)
//   1  fp32, odd offsets : 26 FADD per row and channel  (26 samples)
//   2  u16x2, even offsets: 26 IADD per row and channel (52 samples)
//   3  u16x2, odd offsets : 26 funnel-shift+add (one LEA.HI in SASS) per row and channel (52 samples)
//   4  u16x2, rows alternate even / odd
//   5  u16x2, even offsets with add.u16x2 (SASS VIADD.16x2)
//   6  u16x2, even offsets with mad.lo.u32 x, one, acc (SASS IMAD; ptxas turns add.u32 into IMAD.IADD inside the kernel's bodies)
//   7  u16x2, rows alternate add.u16x2 / funnel-shift+add
// Build + run: nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o /tmp/packed_add paper_1111_6399_b200/microbench/packed_add.cu && /tmp/packed_add
#include <cstdio>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n",cudaGetErrorString(e),__LINE__);return 1;}}while(0)
constexpr int K = 26, D = 4, NW = 32;

template <int MODE> __global__ void __launch_bounds__(384, 1) k(unsigned *out, int nchan) {
    extern __shared__ __align__(16) unsigned sm[];
    for (int i = threadIdx.x; i < 16384; i += blockDim.x) sm[i] = (i * 2654435761u) & 0x00ff00ffu;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned one = nchan > 0 ? 1u : 3u;   // a 1 the compiler cannot see: keeps mode 6 an IMAD
    unsigned acc[D][K];
#pragma unroll
    for (int j = 0; j < D; ++j)
#pragma unroll
        for (int i = 0; i < K; ++i) acc[j][i] = 0;
    unsigned base = (unsigned)__cvta_generic_to_shared(sm) + 4u * (lane * K) + 8u * warp;
    for (int c = 0; c < nchan; ++c) {
        unsigned w[NW];
        const unsigned a = base + ((c & 7) << 12);
#pragma unroll
        for (int m = 0; m < NW / 2; ++m) asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(w[2 * m]), "=r"(w[2 * m + 1]) : "r"(a + 8u * m));
#pragma unroll
        for (int j = 0; j < D; ++j) {
            const int o = j;   // static in-window word offset of row j
            if (MODE == 0) {
#pragma unroll
                for (int i = 0; i < K; i += 2) {
                    unsigned long long p, q;
                    asm("mov.b64 %0, {%1,%2};" : "=l"(p) : "r"(acc[j][i]), "r"(acc[j][i + 1]));
                    asm("mov.b64 %0, {%1,%2};" : "=l"(q) : "r"(w[i + (o & ~1)]), "r"(w[i + (o & ~1) + 1]));
                    asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(p) : "l"(q));
                    asm("mov.b64 {%0,%1}, %2;" : "=r"(acc[j][i]), "=r"(acc[j][i + 1]) : "l"(p));
                }
            } else if (MODE == 1) {
#pragma unroll
                for (int i = 0; i < K; ++i) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(*reinterpret_cast<float *>(&acc[j][i])) : "f"(__uint_as_float(w[i + o])));
            } else if (MODE == 2 || (MODE == 4 && (j & 1) == 0)) {
#pragma unroll
                for (int i = 0; i < K; ++i) asm volatile("add.u32 %0, %0, %1;" : "+r"(acc[j][i]) : "r"(w[i + o]));
            } else if (MODE == 5 || (MODE == 7 && (j & 1) == 0)) {
#pragma unroll
                for (int i = 0; i < K; ++i) asm volatile("add.u16x2 %0, %0, %1;" : "+r"(acc[j][i]) : "r"(w[i + o]));
            } else if (MODE == 6) {
#pragma unroll
                for (int i = 0; i < K; ++i) asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(acc[j][i]) : "r"(w[i + o]), "r"(one));
            } else {
#pragma unroll
                for (int i = 0; i < K; ++i) asm volatile("{.reg .b32 t; shf.r.wrap.b32 t, %1, %2, 16; add.u32 %0, %0, t;}" : "+r"(acc[j][i]) : "r"(w[i + o]), "r"(w[i + o + 1]));
            }
        }
    }
    unsigned s = 0;
#pragma unroll
    for (int j = 0; j < D; ++j)
#pragma unroll
        for (int i = 0; i < K; ++i) s += acc[j][i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

int main() {
    unsigned *d; CK(cudaMalloc(&d, 148 * 384 * 4));
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaDeviceProp pr; cudaGetDeviceProperties(&pr, 0);
    const int nchan = 200000;
    const double clk = pr.clockRate * 1e3;
    printf("SMs %d clock %d kHz, %d channels, 12 warps/SM\n", pr.multiProcessorCount, pr.clockRate, nchan);
    const char *name[8] = {"fp32 even (FADD2)", "fp32 odd (FADD)", "u16x2 even (IADD)", "u16x2 odd (LEA.HI)", "u16x2 mixed", "u16x2 even (VIADD.16x2)", "u16x2 even (IMAD)", "u16x2 mixed VIADD/LEA"};
    for (int mode = 0; mode < 8; ++mode) {
        float ms = 0;
        for (int rep = 0; rep < 3; ++rep) {
            cudaEventRecord(e0);
            if (mode == 0) { CK(cudaFuncSetAttribute(k<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536)); k<0><<<148, 384, 65536>>>(d, nchan); }
            if (mode == 1) { CK(cudaFuncSetAttribute(k<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536)); k<1><<<148, 384, 65536>>>(d, nchan); }
            if (mode == 2) { CK(cudaFuncSetAttribute(k<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536)); k<2><<<148, 384, 65536>>>(d, nchan); }
            if (mode == 3) { CK(cudaFuncSetAttribute(k<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536)); k<3><<<148, 384, 65536>>>(d, nchan); }
            if (mode == 5) { CK(cudaFuncSetAttribute(k<5>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536)); k<5><<<148, 384, 65536>>>(d, nchan); }
            if (mode == 6) { CK(cudaFuncSetAttribute(k<6>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536)); k<6><<<148, 384, 65536>>>(d, nchan); }
            if (mode == 7) { CK(cudaFuncSetAttribute(k<7>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536)); k<7><<<148, 384, 65536>>>(d, nchan); }
            if (mode == 4) { CK(cudaFuncSetAttribute(k<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536)); k<4><<<148, 384, 65536>>>(d, nchan); }
            cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms, e0, e1);
        }
        const double cyc = ms * 1e-3 * clk / nchan;                       // clocks per channel per SM
        const double samples = (mode < 2 ? 1.0 : 2.0) * D * K * 384;       // sample-adds per channel per SM
        printf("mode %d %-20s %8.3f ms  %6.1f clk/channel/SM  %6.1f sample-adds/clk/SM\n", mode, name[mode], ms, cyc, samples / cyc);
    }
    return 0;
}
