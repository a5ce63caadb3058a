// Probe: can a TMA tensor copy (cp.async.bulk.tensor.3d, fp32, no interleave / swizzle) start at ANY element
// of a row, i.e. deliver a window shifted by one sample? No: the copy's first global byte must be 16-byte
// aligned; an inner coordinate that is not a multiple of 4 fp32 elements raises "illegal instruction"
// (profiles/r2_microbench.md). Negative and past-the-end coordinates are fine (zero fill).
// Build + run (one coordinate per process, the error is sticky):
//   nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o /tmp/tma_odd_coord paper_1111_6399_b200/microbench/tma_odd_coord.cu
//   for x in 0 4 -4 3900 1 2 3; do /tmp/tma_odd_coord $x 0; done; /tmp/tma_odd_coord 8 1
// argv: first inner coordinate, 1 = four lanes of a warp each issue a copy (the compiler serialises them)
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
__global__ void k(const __grid_constant__ CUtensorMap tmap, float *out, int x0, int c, int multi) {
    extern __shared__ __align__(1024) unsigned char sm[];
    unsigned base = (unsigned)__cvta_generic_to_shared(sm);
    unsigned bar = base + 8192;
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(multi ? 32 : 1));
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x < (multi ? 32 : 1)) {
        const int lane = threadIdx.x;
        if (lane < 4) {
            asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(1024u) : "memory");
            asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];\n"
                         ::"r"(base + 1024u * lane), "l"(reinterpret_cast<unsigned long long>(&tmap)), "r"(x0 + 256 * lane), "r"(c), "r"(0), "r"(bar) : "memory");
        }
        asm volatile("{.reg .b64 s; mbarrier.arrive.shared::cta.b64 s, [%0];}\n" ::"r"(bar) : "memory");
    }
    asm volatile("{.reg .pred p; W: mbarrier.try_wait.parity.shared::cta.b64 p, [%0], 0; @!p bra W;}\n" ::"r"(bar) : "memory");
    for (int i = threadIdx.x; i < 1024; i += blockDim.x) out[i] = reinterpret_cast<float *>(sm)[i];
}
int main(int argc, char **argv) {
    const int nch = 8; const long long stride = 4096, ns = 4000;
    std::vector<float> h(nch * stride);
    for (size_t i = 0; i < h.size(); ++i) h[i] = (float)i;
    float *d, *o; cudaMalloc(&d, h.size() * 4); cudaMalloc(&o, 4096);
    cudaMemcpy(d, h.data(), h.size() * 4, cudaMemcpyHostToDevice);
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void *fn = nullptr; cudaDriverEntryPointQueryResult q;
    cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
    alignas(64) CUtensorMap tm; memset(&tm, 0, sizeof tm);
    const cuuint64_t dims[3] = {(cuuint64_t)ns, nch, 1}; const cuuint64_t strides[2] = {(cuuint64_t)stride * 4, (cuuint64_t)nch * stride * 4};
    const cuuint32_t box[3] = {256, 1, 1}, es[3] = {1, 1, 1};
    CUresult r = ((encode_fn)fn)(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, d, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                 CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    printf("encode %d q %d\n", (int)r, (int)q);
    cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 16384);
    const int multi = argc > 2 ? atoi(argv[2]) : 0;
        for (int x0 : {argc > 1 ? atoi(argv[1]) : 0}) {
            k<<<1, 128, 16384>>>(tm, o, x0, 3, multi);
            cudaError_t e = cudaDeviceSynchronize();
            float r4[1024]; cudaMemcpy(r4, o, 4096, cudaMemcpyDeviceToHost);
            printf("multi %d x0 %d: %s  out[0]=%g out[5]=%g out[255]=%g out[256]=%g (want %g)\n", multi, x0, cudaGetErrorString(e), r4[0], r4[5], r4[255], r4[256], (double)(3 * stride + x0));
            if (e != cudaSuccess) return 1;
        }
}
