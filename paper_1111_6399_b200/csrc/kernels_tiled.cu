// kernels_tiled.cu — the NAIVE cross-check kernel and the generic TILED kernel.
//
// Both compute out[d][t] = sum_c in[c][t + s(c,d)] (§2) for every dtype and every plan.
// TILED follows the paper's Fig. 2: a CTA owns a rectangle of (DM, t) space, each
// thread keeps several accumulators in registers, and the (f,t) data a rectangle needs is fetched
// once per CTA and reused by all its DM rows. On Fermi that reuse came from L1 cache-lines; here
// the channel's time window [t0 + s(c,d_first), t0 + T + s(c,d_last)] is staged explicitly into a
// double-buffered shared-memory ring with 16-byte cp.async.
// It reads one shared-memory word per add, so it tops out near 25 % of the FP32 add peak; the
// SUBBAND kernel (subband.cu) is the fast path, this one is the always-applicable one.
#include <cuda_fp16.h>

#include <algorithm>
#include <cstdint>

#include "plan.h"

namespace {

// ------------------------------------------------------------------ element access
template <typename TIN> struct Elem;
template <> struct Elem<uint8_t> {
    using Acc = int;
    static __device__ __forceinline__ int load(const uint8_t *p) { return (int)*p; }
};
template <> struct Elem<__half> {
    using Acc = float;
    static __device__ __forceinline__ float load(const __half *p) { return __half2float(*p); }
};
template <> struct Elem<float> {
    using Acc = float;
    static __device__ __forceinline__ float load(const float *p) { return *p; }
};

// ------------------------------------------------------------------ NAIVE
// One thread per (d, t); every term read from global memory through L1. The parity tests check it
// against the oracle on whole outputs, then use it as the full-size cross-check for the others.
template <typename TIN>
__global__ void __launch_bounds__(256) dedisp_naive_kernel(const TIN *__restrict__ in, long long in_stride,
                                                           typename Elem<TIN>::Acc *__restrict__ out,
                                                           long long out_stride, long long nsamp_out,
                                                           const int *__restrict__ shifts, int nchans, int ndm,
                                                           long long in_beam, long long out_beam) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int d = blockIdx.y;
    if (t >= nsamp_out) return;
    in += (size_t)blockIdx.z * in_beam;
    out += (size_t)blockIdx.z * out_beam;
    typename Elem<TIN>::Acc acc = 0;
    for (int c = 0; c < nchans; ++c) {
        const int s = __ldg(shifts + (size_t)c * ndm + d);
        acc += Elem<TIN>::load(in + (size_t)c * in_stride + t + s);
    }
    out[(size_t)d * out_stride + t] = acc;
}

// ------------------------------------------------------------------ TILED
constexpr int TILED_THREADS = 256;
constexpr int TILED_WARPS = 8;
constexpr int TILED_KT = 16;                 // samples per thread, interleaved by 32
constexpr int TILED_T = 32 * TILED_KT;       // 512 output samples per CTA
constexpr int TILED_SMEM_BUDGET = 96 * 1024; // both stages; leaves room for 2 CTAs per SM

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem, int src_bytes) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(sa), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

// CTA: 8 warps; warp w owns DM rows d0 + w*DT .. +DT-1; lane l owns samples t0 + l + 32k, k < KT.
// Shared memory: 2 stages x cb slots of slot_bytes raw input bytes + 2 x cb x (8*DT) int offsets.
template <typename TIN, int DT>
__global__ void __launch_bounds__(TILED_THREADS, 2)
dedisp_tiled_kernel(const TIN *__restrict__ in, long long in_stride, long long in_total_elems,
                    typename Elem<TIN>::Acc *__restrict__ out, long long out_stride, long long nsamp_out,
                    const int *__restrict__ shifts, int nchans, int ndm, int slot_bytes, int cb,
                    long long in_beam, long long out_beam) {
    using Acc = typename Elem<TIN>::Acc;
    constexpr int ROWS = TILED_WARPS * DT;
    in += (size_t)blockIdx.z * in_beam;
    out += (size_t)blockIdx.z * out_beam;
    extern __shared__ __align__(16) unsigned char smem[];
    unsigned char *sdata = smem;                                        // [2][cb][slot_bytes]
    int *soff = reinterpret_cast<int *>(smem + (size_t)2 * cb * slot_bytes);  // [2][cb][ROWS]

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int d0 = blockIdx.y * ROWS;
    const int dlast = min(d0 + ROWS, ndm) - 1;
    const long long t0 = (long long)blockIdx.x * TILED_T;
    const unsigned long long in_base = (unsigned long long)in;
    const unsigned long long in_end = in_base + (unsigned long long)in_total_elems * sizeof(TIN);

    Acc acc[DT][TILED_KT];
#pragma unroll
    for (int j = 0; j < DT; ++j)
#pragma unroll
        for (int k = 0; k < TILED_KT; ++k) acc[j][k] = 0;

    const int nstages = (nchans + cb - 1) / cb;

    auto issue_stage = [&](int stage) {
        const int buf = stage & 1;
        for (int ch = 0; ch < cb; ++ch) {
            const int c = stage * cb + ch;
            if (c >= nchans) break;
            const int *srow = shifts + (size_t)c * ndm;
            const int smin = __ldg(srow + d0);
            const int smax = __ldg(srow + dlast);
            // window start as a byte address, aligned down to 16 B; the remainder joins the offsets
            const unsigned long long a0 =
                in_base + ((unsigned long long)c * in_stride + t0 + smin) * sizeof(TIN);
            const unsigned long long a0al = a0 & ~15ull;
            const int rem = (int)(a0 - a0al) / (int)sizeof(TIN);
            const int nbytes = (int)(a0 - a0al) + (TILED_T + smax - smin) * (int)sizeof(TIN);
            const int nchunks = (nbytes + 15) >> 4;
            unsigned char *slot = sdata + ((size_t)buf * cb + ch) * slot_bytes;
            for (int i = tid; i < nchunks; i += TILED_THREADS) {
                const unsigned long long ga = a0al + (unsigned long long)i * 16;
                long long valid = (long long)in_end - (long long)ga;
                valid = valid < 0 ? 0 : (valid > 16 ? 16 : valid);
                cp_async16(slot + i * 16, (const void *)(valid ? ga : in_base), (int)valid);
            }
            if (tid < ROWS) {
                const int d = min(d0 + tid, ndm - 1);
                soff[((size_t)buf * cb + ch) * ROWS + tid] = __ldg(srow + d) - smin + rem;
            }
        }
        cp_async_commit();
    };

    issue_stage(0);
    for (int stage = 0; stage < nstages; ++stage) {
        if (stage + 1 < nstages) {
            issue_stage(stage + 1);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        __syncthreads();
        const int buf = stage & 1;
        const int nch = min(cb, nchans - stage * cb);
        for (int ch = 0; ch < nch; ++ch) {
            const TIN *slot = reinterpret_cast<const TIN *>(sdata + ((size_t)buf * cb + ch) * slot_bytes);
            const int *offs = soff + ((size_t)buf * cb + ch) * ROWS + warp * DT;
#pragma unroll
            for (int j = 0; j < DT; ++j) {
                const TIN *p = slot + offs[j] + lane;
#pragma unroll
                for (int k = 0; k < TILED_KT; ++k) acc[j][k] += Elem<TIN>::load(p + 32 * k);
            }
        }
        __syncthreads();
    }

#pragma unroll
    for (int j = 0; j < DT; ++j) {
        const int d = d0 + warp * DT + j;
        if (d >= ndm) continue;
        Acc *orow = out + (size_t)d * out_stride;
#pragma unroll
        for (int k = 0; k < TILED_KT; ++k) {
            const long long t = t0 + lane + 32 * k;
            if (t < nsamp_out) orow[t] = acc[j][k];
        }
    }
}

template <typename TIN>
cudaError_t launch_tiled_t(const dedisp_plan *p, const void *d_in, long long in_stride, long long nsamp_out,
                           void *d_out, long long out_stride, Batch b, cudaStream_t st) {
    using Acc = typename Elem<TIN>::Acc;
    const TiledGeom &g = p->tiled;
    const int rows = TILED_WARPS * g.dt;
    dim3 grid((unsigned)((nsamp_out + TILED_T - 1) / TILED_T), (unsigned)((p->ndm + rows - 1) / rows), (unsigned)b.n);
    const size_t smem = (size_t)2 * g.cb * g.slot_bytes + (size_t)2 * g.cb * rows * sizeof(int);
    const long long in_total = (long long)(p->nchans - 1) * in_stride + nsamp_out + p->maxshift;
    auto go = [&](auto kern) -> cudaError_t {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        kern<<<grid, TILED_THREADS, smem, st>>>((const TIN *)d_in, in_stride, in_total, (Acc *)d_out, out_stride,
                                                nsamp_out, p->d_shifts, p->nchans, p->ndm, g.slot_bytes, g.cb,
                                                b.in_stride, b.out_stride);
        return cudaGetLastError();
    };
    switch (g.dt) {
        case 4: return go(dedisp_tiled_kernel<TIN, 4>);
        case 2: return go(dedisp_tiled_kernel<TIN, 2>);
        default: return go(dedisp_tiled_kernel<TIN, 1>);
    }
}

template <typename TIN>
cudaError_t launch_naive_t(const dedisp_plan *p, const void *d_in, long long in_stride, long long nsamp_out,
                           void *d_out, long long out_stride, Batch b, cudaStream_t st) {
    using Acc = typename Elem<TIN>::Acc;
    dim3 grid((unsigned)((nsamp_out + 255) / 256), (unsigned)p->ndm, (unsigned)b.n);
    dedisp_naive_kernel<TIN><<<grid, 256, 0, st>>>((const TIN *)d_in, in_stride, (Acc *)d_out, out_stride,
                                                    nsamp_out, p->d_shifts, p->nchans, p->ndm, b.in_stride, b.out_stride);
    return cudaGetLastError();
}

}  // namespace

// Pick the largest DM tile (8*dt rows) whose widest channel window fits the slot budget.
void tiled_choose_geom(dedisp_plan *p) {
    const int esize = dtype_esize(p->dtype);
    p->tiled = TiledGeom();
    for (int dt : {4, 2, 1}) {
        const int rows = TILED_WARPS * dt;
        long long spread = 0;
        for (int c = 0; c < p->nchans; ++c) {
            const int32_t *row = p->shifts.data() + (size_t)c * p->ndm;
            for (int d0 = 0; d0 < p->ndm; d0 += rows) {
                const int dl = std::min(d0 + rows, p->ndm) - 1;
                spread = std::max<long long>(spread, (long long)row[dl] - row[d0]);
            }
        }
        const long long slot = (((TILED_T + spread) * esize + 16 + 15) / 16) * 16;  // +16: alignment remainder
        const long long per_chan = 2 * (slot + (long long)rows * 4);
        if (per_chan > TILED_SMEM_BUDGET) continue;
        p->tiled.ok = true;
        p->tiled.dt = dt;
        p->tiled.slot_bytes = (int)slot;
        p->tiled.cb = (int)std::min<long long>(8, TILED_SMEM_BUDGET / per_chan);
        return;
    }
}

cudaError_t launch_naive(const dedisp_plan *p, const void *d_in, long long in_stride, long long nsamp_out,
                         void *d_out, long long out_stride, Batch b, cudaStream_t st) {
    switch (p->dtype) {
        case DEDISP_U8: return launch_naive_t<uint8_t>(p, d_in, in_stride, nsamp_out, d_out, out_stride, b, st);
        case DEDISP_F16: return launch_naive_t<__half>(p, d_in, in_stride, nsamp_out, d_out, out_stride, b, st);
        default: return launch_naive_t<float>(p, d_in, in_stride, nsamp_out, d_out, out_stride, b, st);
    }
}

cudaError_t launch_tiled(const dedisp_plan *p, const void *d_in, long long in_stride, long long nsamp_out,
                         void *d_out, long long out_stride, Batch b, cudaStream_t st) {
    switch (p->dtype) {
        case DEDISP_U8: return launch_tiled_t<uint8_t>(p, d_in, in_stride, nsamp_out, d_out, out_stride, b, st);
        case DEDISP_F16: return launch_tiled_t<__half>(p, d_in, in_stride, nsamp_out, d_out, out_stride, b, st);
        default: return launch_tiled_t<float>(p, d_in, in_stride, nsamp_out, d_out, out_stride, b, st);
    }
}
