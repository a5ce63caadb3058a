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
// Two HBM-bound kernels: row statistics (one read of the block) and boxcar + threshold (one more read,
// plus a halo of 2^(nwidths-1) - 1 samples per tile); roofline = 2 x block bytes / HBM bandwidth.
#include <cstdint>
#include <type_traits>

#include "plan.h"

namespace {

constexpr int DET_THREADS = 256;
constexpr int DET_PER = 8;                          // samples per thread and tile
constexpr int DET_TILE = DET_THREADS * DET_PER;     // 2048 samples per CTA tile
constexpr int DET_MAXW = 1 << (DEDISP_DETECT_MAX_WIDTHS - 1);

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

template <typename T>
__global__ void __launch_bounds__(DET_THREADS) dedisp_detect_boxcar_kernel(const T *__restrict__ x, long long stride, long long n, int nwidths,
                                                                             double threshold, const unsigned long long *__restrict__ stats,
                                                                             dedisp_candidate *__restrict__ cands, long long max_cands,
                                                                             unsigned long long *__restrict__ count) {
    __shared__ T buf[2][DET_TILE + DET_MAXW];
    const int row_i = blockIdx.y;
    // mean and variance exactly as the definition orders them (explicitly rounded double operations)
    double mu, var;
    if constexpr (sizeof(T) == 4 && !std::is_floating_point<T>::value) {
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
    const T *row = x + (size_t)row_i * stride;
    const long long t0 = (long long)blockIdx.x * DET_TILE;
    const int halo = (1 << (nwidths - 1)) - 1;
    const int nload = (int)min((long long)DET_TILE + halo, n - t0);     // samples of the row available from t0
    for (int i = threadIdx.x; i < DET_TILE + halo; i += DET_THREADS) buf[0][i] = i < nload ? row[t0 + i] : (T)0;
    __syncthreads();
    // snr is monotone in y (rw > 0, every operation rounds monotonically), so "snr >= threshold" is "y >= Y_w"
    // for the smallest representable Y_w that passes: thread k finds Y_w for width 2^k once per CTA, the scan
    // then compares in the row's own type and evaluates the double expression only for the rare candidates
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
    int cur = 0;
    for (int k = 0, w = 1; k < nwidths; ++k, w *= 2) {
        if (k > 0) {   // y_w[i] = y_{w/2}[i] + y_{w/2}[i + w/2], wherever the wider window still fits the loaded span
            const int h = w / 2, lim = DET_TILE + halo - w + 1;
            for (int i = threadIdx.x; i < lim; i += DET_THREADS) buf[cur ^ 1][i] = (T)(buf[cur][i] + buf[cur][i + h]);
            cur ^= 1;
            __syncthreads();
        }
        if (ynone[k]) continue;
        const T crit = ycrit[k];
        for (int i = threadIdx.x; i < DET_TILE; i += DET_THREADS) {
            if (t0 + i + w > n) break;                                  // the window must lie inside the row
            const T y = buf[cur][i];
            if (y >= crit) {
                const double wm = __dmul_rn((double)w, mu);
                const double rw = __ddiv_rn(1.0, __dmul_rn(sd, __dsqrt_rn((double)w)));
                const double snr = __dmul_rn(__dsub_rn((double)y, wm), rw);
                if (snr >= threshold) {                                // always true; kept as the definition's own test
                    const unsigned long long slot = atomicAdd(count, 1ull);
                    if ((long long)slot < max_cands) {
                        dedisp_candidate c;
                        c.dm_index = row_i; c.width = w; c.t = t0 + i; c.snr = snr;
                        cands[slot] = c;
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
    const dim3 g1((unsigned)((nsamp + DET_TILE * 8 - 1) / (DET_TILE * 8)), (unsigned)ndm), g2((unsigned)((nsamp + DET_TILE - 1) / DET_TILE), (unsigned)ndm);
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
