// detect.cu — detection behind the de-dispersion hot path ("detect
// millisecond radio bursts ... in real-time", "detection of interesting signals"), so that the
// de-dispersed block (c5: 4.3 GB per chunk) never has to leave the GPU. The paper gives no algorithm; the
// definition is DESIGN.md reading R16 (see include/dedisp.h, dedisp_detect):
//
//   per DM row: S1 = sum x, S2 = sum x^2 (exact 64-bit integers for int32 rows, double for fp32 rows),
//   mu = S1/N, var = S2/N - mu^2; boxcar sums y_w by doubling (w = 1, 2, 4, ...) in the row's own
//   arithmetic; snr_w[t] = (y_w[t] - w mu) * (1 / (sqrt(var) sqrt(w))) in IEEE double with explicitly
//   rounded operations (no contraction), so that integer rows give bit-identical S/N on CPU and GPU;
//   every (row, w, t) with snr >= threshold is appended to a candidate list through one atomic counter.
//
// Two HBM-bound kernels: row statistics (one read of the block) and boxcar + threshold (one more read;
// neighbouring warp segments overlap by the largest width, served by L1/L2); roofline = 2 x block bytes /
// HBM bandwidth.
#include <cstdint>
#include <mutex>
#include <type_traits>

#include "plan.h"

namespace {

constexpr int DET_THREADS = 256;
constexpr int DET_PER = 8;                          // samples per thread and tile
constexpr int DET_TILE = DET_THREADS * DET_PER;     // 2048 samples per CTA tile
constexpr int DET_MAXW = 1 << (DEDISP_DETECT_MAX_WIDTHS - 1);
constexpr int DET_SEGS = 8;                         // boxcar kernel: 256-sample segments per warp
inline int det_own(int nwidths) { return 256 - ((((1 << (nwidths - 1)) - 1) + 7) & ~7); }   // positions a 256-sample warp segment owns
static_assert(DET_MAXW <= 128, "a segment must own at least half of its samples");

template <typename T>
__global__ void __launch_bounds__(DET_THREADS) dedisp_detect_stats_kernel(const T *__restrict__ x, long long stride, long long n,
                                                                            unsigned long long *__restrict__ stats) {
    // grid: (chunks of the row, rows). stats[row] = {S1, S2}: int64 bit patterns (exact, order-free atomics) for
    // integer rows, double bit patterns for float rows
    const T *row = x + (size_t)blockIdx.y * stride;
    const long long t0 = (long long)blockIdx.x * (DET_TILE * 8);
    const long long t1 = min(n, t0 + (long long)DET_TILE * 8);
    if constexpr (sizeof(T) == 4 && !std::is_floating_point<T>::value) {
        long long s1 = 0, s2 = 0;
        for (long long t = t0 + threadIdx.x; t < t1; t += DET_THREADS) { const long long v = row[t]; s1 += v; s2 += v * v; }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { s1 += __shfl_xor_sync(0xffffffffu, s1, o); s2 += __shfl_xor_sync(0xffffffffu, s2, o); }
        if ((threadIdx.x & 31) == 0) {
            atomicAdd(stats + 2 * blockIdx.y, (unsigned long long)s1);
            atomicAdd(stats + 2 * blockIdx.y + 1, (unsigned long long)s2);
        }
    } else {
        double s1 = 0.0, s2 = 0.0;
        for (long long t = t0 + threadIdx.x; t < t1; t += DET_THREADS) { const double v = (double)row[t]; s1 += v; s2 += v * v; }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { s1 += __shfl_xor_sync(0xffffffffu, s1, o); s2 += __shfl_xor_sync(0xffffffffu, s2, o); }
        if ((threadIdx.x & 31) == 0) {
            atomicAdd(reinterpret_cast<double *>(stats) + 2 * blockIdx.y, s1);
            atomicAdd(reinterpret_cast<double *>(stats) + 2 * blockIdx.y + 1, s2);
        }
    }
}

// Boxcar + threshold. A warp owns a segment of 256 consecutive samples of one row, 8 per lane in registers;
// the next width comes from the current one by y_2w[p] = y_w[p] + y_w[p + w], where p + w lives w/8 lanes
// further (a shuffle) or, for w < 8, partly in the lane's own registers. Segments overlap by H = the largest
// width rounded up to 8, so that every position a segment owns (the first 256 - H) finds all its windows
// inside the segment. Because S/N is monotone in the window sum (rw > 0, every operation rounds
// monotonically), "snr >= threshold" is "y >= Y_w" for the smallest representable Y_w that passes: thread k
// finds Y_w for width 2^k once per CTA with the exact double expression, the scan compares in the row's
// own type (one SETP per sample and width, OR-ed into one predicate per lane) and evaluates the double S/N
// only for the rare hits, which one atomic counter compacts into the caller's list.
template <typename T>
__global__ void __launch_bounds__(DET_THREADS) dedisp_detect_boxcar_kernel(const T *__restrict__ x, long long stride, long long n, int nwidths,
                                                                             double threshold, const unsigned long long *__restrict__ stats,
                                                                             dedisp_candidate *__restrict__ cands, long long max_cands,
                                                                             unsigned long long *__restrict__ count) {
    const int row_i = blockIdx.y;
    // mean and variance exactly as the definition orders them (explicitly rounded double operations)
    double mu, var;
    if constexpr (!std::is_floating_point<T>::value) {
        const long long s1 = (long long)stats[2 * row_i], s2 = (long long)stats[2 * row_i + 1];
        mu = __ddiv_rn((double)s1, (double)n);
        var = __dsub_rn(__ddiv_rn((double)s2, (double)n), __dmul_rn(mu, mu));
    } else {
        const double s1 = reinterpret_cast<const double *>(stats)[2 * row_i], s2 = reinterpret_cast<const double *>(stats)[2 * row_i + 1];
        mu = __ddiv_rn(s1, (double)n);
        var = __dsub_rn(__ddiv_rn(s2, (double)n), __dmul_rn(mu, mu));
    }
    if (!(var > 0.0)) return;
    const double sd = __dsqrt_rn(var);
    __shared__ T ycrit[DEDISP_DETECT_MAX_WIDTHS];
    __shared__ int ynone[DEDISP_DETECT_MAX_WIDTHS];
    if (threadIdx.x < nwidths) {
        const int w = 1 << threadIdx.x;
        const double wm = __dmul_rn((double)w, mu);
        const double rw = __ddiv_rn(1.0, __dmul_rn(sd, __dsqrt_rn((double)w)));
        auto pass = [&](double y) { return __dmul_rn(__dsub_rn(y, wm), rw) >= threshold; };
        const double guess = threshold / rw + wm;
        int none = 0;
        T crit;
        if constexpr (std::is_floating_point<T>::value) {
            float y = guess > 3.0e38 ? 3.0e38f : guess < -3.0e38 ? -3.0e38f : (float)guess;
            if (!(guess == guess)) none = 1;
            for (int i = 0; i < 64 && !none && y > -3.0e38f && pass((double)nextafterf(y, -INFINITY)); ++i) y = nextafterf(y, -INFINITY);
            for (int i = 0; i < 64 && !none && !pass((double)y); ++i) { if (y >= 3.0e38f) { none = 1; break; } y = nextafterf(y, INFINITY); }
            if (!none && !pass((double)y)) none = 1;
            crit = y;
        } else {
            long long y = guess > 2147483647.0 ? 2147483647ll : guess < -2147483648.0 ? -2147483648ll : (long long)floor(guess);
            if (!(guess == guess)) none = 1;
            for (int i = 0; i < 64 && !none && y > -2147483648ll && pass((double)(y - 1)); ++i) --y;
            for (int i = 0; i < 64 && !none && !pass((double)y); ++i) { if (y >= 2147483647ll) { none = 1; break; } ++y; }
            if (!none && !pass((double)y)) none = 1;
            crit = (T)y;
        }
        ycrit[threadIdx.x] = crit;
        ynone[threadIdx.x] = none;
    }
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int H = ((1 << (nwidths - 1)) - 1 + 7) & ~7;              // overlap between neighbouring segments
    const int own = 256 - H;                                       // positions a segment owns
    const T *row = x + (size_t)row_i * stride;
#pragma unroll 1
    for (int rep = 0; rep < DET_SEGS; ++rep) {                     // DET_SEGS segments per warp: the critical values are found once per CTA
    const long long t0 = (((long long)blockIdx.x * DET_SEGS + rep) * (DET_THREADS / 32) + (threadIdx.x >> 5)) * own;
    if (t0 >= n) return;
    T v[8];
    const T *src = row + t0 + 8 * lane;
    if (t0 + 256 <= n && (reinterpret_cast<uintptr_t>(src) & 15) == 0) {   // interior segment, 16-byte aligned: two vector loads
        const uint4 a = __ldg(reinterpret_cast<const uint4 *>(src)), b = __ldg(reinterpret_cast<const uint4 *>(src) + 1);
        const unsigned raw[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if constexpr (std::is_floating_point<T>::value) v[i] = __uint_as_float(raw[i]);
            else v[i] = (T)raw[i];
        }
    } else {
#pragma unroll
        for (int i = 0; i < 8; ++i) { const long long t = t0 + 8 * lane + i; v[i] = t < n ? row[t] : (T)0; }
    }
#pragma unroll
    for (int k = 0; k < DEDISP_DETECT_MAX_WIDTHS; ++k) {
        if (k >= nwidths) break;
        const int w = 1 << k;
        if (k > 0) {                                               // y_w[p] = y_h[p] + y_h[p + h], h = w / 2
            constexpr int KH = 1;
            (void)KH;
            const int h = w / 2;
            T u[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                T partner;
                if (h < 8) partner = i + h < 8 ? v[(i + h) & 7] : __shfl_down_sync(0xffffffffu, v[(i + h) & 7], 1);
                else partner = __shfl_down_sync(0xffffffffu, v[i], h / 8);
                u[i] = (T)(v[i] + partner);
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) v[i] = u[i];
        }
        if (ynone[k]) continue;
        const T crit = ycrit[k];
        bool hit = false;
#pragma unroll
        for (int i = 0; i < 8; ++i) hit |= v[i] >= crit;
        if (hit) {
            const double wm = __dmul_rn((double)w, mu);
            const double rw = __ddiv_rn(1.0, __dmul_rn(sd, __dsqrt_rn((double)w)));
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int pos = 8 * lane + i;
                const long long t = t0 + pos;
                if (v[i] >= crit && pos < own && t + w <= n) {       // owned position, window inside the row
                    const double snr = __dmul_rn(__dsub_rn((double)v[i], wm), rw);
                    if (snr >= threshold) {                         // always true; kept as the definition's own test
                        const unsigned long long slot = atomicAdd(count, 1ull);
                        if ((long long)slot < max_cands) {
                            dedisp_candidate c;
                            c.dm_index = row_i; c.width = w; c.t = t; c.snr = snr;
                            cands[slot] = c;
                        }
                    }
                }
            }
        }
    }
    }
}

}  // namespace

extern "C" {

long long dedisp_detect_workspace_bytes(int ndm) { return ndm < 0 ? -1 : (long long)ndm * 16 + 8; }

int dedisp_detect(const void *d_block, int block_is_float, int ndm, long long nsamp, long long stride, int nwidths, double threshold,
                  dedisp_candidate *d_cands, long long max_cands, void *d_work, void *stream) {
    if (!d_block || !d_work || ndm < 1 || ndm > 65535 || nsamp < 1 || stride < nsamp || max_cands < 0 || (max_cands && !d_cands)) return DEDISP_EINVAL;
    if (nwidths < 1 || nwidths > DEDISP_DETECT_MAX_WIDTHS || ((uintptr_t)d_work & 7)) return DEDISP_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long *count = reinterpret_cast<unsigned long long *>(d_work);
    unsigned long long *stats = count + 1;
    cudaError_t e = cudaMemsetAsync(d_work, 0, (size_t)ndm * 16 + 8, st);
    if (e != cudaSuccess) return DEDISP_ECUDA;
    const dim3 g1((unsigned)((nsamp + DET_TILE * 8 - 1) / (DET_TILE * 8)), (unsigned)ndm), g2((unsigned)((nsamp + (long long)det_own(nwidths) * (DET_THREADS / 32) * DET_SEGS - 1) / ((long long)det_own(nwidths) * (DET_THREADS / 32) * DET_SEGS)), (unsigned)ndm);
    if (block_is_float) {
        dedisp_detect_stats_kernel<float><<<g1, DET_THREADS, 0, st>>>((const float *)d_block, stride, nsamp, stats);
        dedisp_detect_boxcar_kernel<float><<<g2, DET_THREADS, 0, st>>>((const float *)d_block, stride, nsamp, nwidths, threshold, stats, d_cands, max_cands, count);
    } else {
        dedisp_detect_stats_kernel<int><<<g1, DET_THREADS, 0, st>>>((const int *)d_block, stride, nsamp, stats);
        dedisp_detect_boxcar_kernel<int><<<g2, DET_THREADS, 0, st>>>((const int *)d_block, stride, nsamp, nwidths, threshold, stats, d_cands, max_cands, count);
    }
    return cudaGetLastError() == cudaSuccess ? DEDISP_OK : DEDISP_ECUDA;
}

}  // extern "C"

// =====================================================================================
// dedisp_detect_static: the same two kernels for callers that cannot provide (or allocate) scratch memory
// =====================================================================================
namespace {

// Scratch of dedisp_detect_static: {S1, S2} of every DM row. 128 KB that every GPU which loads the library holds
// until the process exits. In HOST code this name is a host-side stand-in, not a device address: the address the
// kernels get is looked up once per device with cudaGetSymbolAddress (det_static_scratch below).
static __device__ __align__(256) unsigned long long det_static_stats[2 * DEDISP_DETECT_STATIC_MAX_NDM];

constexpr int DET_MAX_DEVICES = 64;
std::mutex det_static_mu;
unsigned long long *det_static_addr[DET_MAX_DEVICES];   // device address of det_static_stats on device i, NULL: not looked up yet

// Device address of the static scratch on the CURRENT device (set-up: once per device, with that device current).
cudaError_t det_static_scratch(unsigned long long **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= DET_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(det_static_mu);
    if (!det_static_addr[dev]) {
        unsigned long long *ptr = nullptr;
        e = cudaGetSymbolAddress((void **)&ptr, det_static_stats);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        det_static_addr[dev] = ptr;
    }
    *out = det_static_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int dedisp_detect_static(const void *d_block, int block_is_float, int ndm, long long nsamp, long long stride, int nwidths,
                                    double threshold, dedisp_candidate *d_cands, long long max_cands, unsigned long long *d_count,
                                    void *stream) {
    if (!d_block || !d_count || ((uintptr_t)d_count & 7) || ndm < 1 || nsamp < 1 || stride < nsamp || max_cands < 0 || (max_cands && !d_cands))
        return DEDISP_EINVAL;
    if (nwidths < 1 || nwidths > DEDISP_DETECT_MAX_WIDTHS) return DEDISP_EINVAL;
    if (ndm > DEDISP_DETECT_STATIC_MAX_NDM) return DEDISP_ETOOLARGE;   // the static scratch holds no more rows
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long *stats = nullptr;
    if (det_static_scratch(&stats) != cudaSuccess) return DEDISP_ECUDA;
    // the array keeps the last call's sums, and the sums are accumulated with atomics: clear the rows of this call
    cudaError_t e = cudaMemsetAsync(stats, 0, (size_t)ndm * 16, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(d_count, 0, 8, st);
    if (e != cudaSuccess) return DEDISP_ECUDA;
    const long long per2 = (long long)det_own(nwidths) * (DET_THREADS / 32) * DET_SEGS;
    const dim3 g1((unsigned)((nsamp + DET_TILE * 8 - 1) / (DET_TILE * 8)), (unsigned)ndm), g2((unsigned)((nsamp + per2 - 1) / per2), (unsigned)ndm);
    if (block_is_float) {
        dedisp_detect_stats_kernel<float><<<g1, DET_THREADS, 0, st>>>((const float *)d_block, stride, nsamp, stats);
        dedisp_detect_boxcar_kernel<float><<<g2, DET_THREADS, 0, st>>>((const float *)d_block, stride, nsamp, nwidths, threshold, stats, d_cands, max_cands, d_count);
    } else {
        dedisp_detect_stats_kernel<int><<<g1, DET_THREADS, 0, st>>>((const int *)d_block, stride, nsamp, stats);
        dedisp_detect_boxcar_kernel<int><<<g2, DET_THREADS, 0, st>>>((const int *)d_block, stride, nsamp, nwidths, threshold, stats, d_cands, max_cands, d_count);
    }
    return cudaGetLastError() == cudaSuccess ? DEDISP_OK : DEDISP_ECUDA;
}
