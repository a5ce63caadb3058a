// Stronger CPU baseline for bench.py - a REPORTING baseline, not the product and
// not the oracle. The modern counterpart of the paper's second algorithm (section 4: a
// "vector-parallel" CPU kernel "designed with maximum cache-line usage in mind", SSE/AVX intrinsics on the
// paper's Xeon / Sandy Bridge): brute-force de-dispersion, threaded over DM rows, blocked in time so that a
// row's accumulator tile stays in L1, with the inner loop `acc[t] += in[c][t + s]` over contiguous samples
// left to the compiler's vectoriser (-O3 -march=native: AVX-512 / AVX2 adds, widening u8 -> i32 loads).
// Every (d, c, t) term is added, nothing is shared between trials. Own delay computation (same expression
// as DESIGN.md reading R4); checked against the oracle in tests/test_cpu_baseline.py.
//
// Build: g++ -O3 -march=native -std=c++17 -ffp-contract=off -fPIC -shared -pthread (baseline_cpu/__init__.py).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <thread>
#include <vector>

namespace {

constexpr long long TILE = 8192;   // accumulator tile: 32 KB of int32 / float, L1-resident

long long delay(double fch1, double foff, double tsamp, double dm, int c) {
    const double f = fch1 + c * foff;
    return (long long)std::floor(((4.148808e3 * dm) * (1.0 / (f * f) - 1.0 / (fch1 * fch1))) / tsamp + 0.5);
}

template <typename TIN, typename TACC>
void rows_range(int nchans, const std::vector<long long>& shifts, int ndm, const TIN* in, long long in_stride,
                long long nsamp_out, TACC* out, int d0, int d1) {
    std::vector<TACC> acc((size_t)TILE);
    for (int d = d0; d < d1; ++d)
        for (long long t0 = 0; t0 < nsamp_out; t0 += TILE) {
            const long long n = std::min(TILE, nsamp_out - t0);
            std::fill(acc.begin(), acc.begin() + n, (TACC)0);
            for (int c = 0; c < nchans; ++c) {
                const TIN* row = in + (long long)c * in_stride + t0 + shifts[(size_t)c * ndm + d];
                TACC* a = acc.data();
                for (long long t = 0; t < n; ++t) a[t] += (TACC)row[t];
            }
            std::copy(acc.begin(), acc.begin() + n, out + (long long)d * nsamp_out + t0);
        }
}

template <typename TIN, typename TACC>
int run(int nchans, double fch1, double foff, double tsamp, const double* dm, int ndm, const TIN* in, long long in_stride,
        long long nsamp_in, long long nsamp_out, TACC* out, int nthreads) {
    if (nchans < 1 || ndm < 1 || nsamp_out < 1 || !in || !out || nthreads < 1) return 1;
    std::vector<long long> shifts((size_t)nchans * ndm);
    for (int c = 0; c < nchans; ++c)
        for (int d = 0; d < ndm; ++d) {
            const long long s = delay(fch1, foff, tsamp, dm[d], c);
            if (s < 0 || s + nsamp_out > nsamp_in) return 2;
            shifts[(size_t)c * ndm + d] = s;
        }
    nthreads = std::min(nthreads, ndm);
    std::vector<std::thread> th;
    for (int i = 0; i < nthreads; ++i) {
        const int d0 = (int)((long long)ndm * i / nthreads), d1 = (int)((long long)ndm * (i + 1) / nthreads);
        th.emplace_back([=, &shifts] { rows_range<TIN, TACC>(nchans, shifts, ndm, in, in_stride, nsamp_out, out, d0, d1); });
    }
    for (auto& t : th) t.join();
    return 0;
}

}  // namespace

extern "C" {
// out[d][t] for the DM list given (all of it); u8 -> int32, f32 -> float (fp32 accumulation, channel order).
int cpu_vec_dedisperse_u8(int nchans, double fch1, double foff, double tsamp, const double* dm, int ndm, const uint8_t* in,
                          long long in_stride, long long nsamp_in, long long nsamp_out, int32_t* out, int nthreads) {
    return run<uint8_t, int32_t>(nchans, fch1, foff, tsamp, dm, ndm, in, in_stride, nsamp_in, nsamp_out, out, nthreads);
}
int cpu_vec_dedisperse_f32(int nchans, double fch1, double foff, double tsamp, const double* dm, int ndm, const float* in,
                           long long in_stride, long long nsamp_in, long long nsamp_out, float* out, int nthreads) {
    return run<float, float>(nchans, fch1, foff, tsamp, dm, ndm, in, in_stride, nsamp_in, nsamp_out, out, nthreads);
}
}
