// ORACLE — test infrastructure, NOT the product.
//
// Plain CPU statement of the step behind the de-dispersion hot path (
// PAPER.md:18 "detect millisecond radio bursts ... in real-time", "detection of interesting
// signals"). The paper names the step and gives no algorithm, so the definition below is this build's own
// (reading R16); this file states it step by step, in the order given there. It shares no code
// with paper_1111_6399_b200/csrc/ nor with the other oracle files.
//
// For every DM row x[0..N) of the de-dispersed block (int32 or float32):
//   1. S1 = sum x[t], S2 = sum x[t]^2            (int rows: exact 64-bit integers; float rows: double,
//                                                  t ascending), mu = S1/N, var = S2/N - mu*mu (double).
//      A row with var <= 0 yields no candidates.
//   2. boxcar sums of width w = 1, 2, 4, ..., 2^(nwidths-1) by doubling, in the row's own arithmetic
//      (int32 adds / fp32 adds): y_1[t] = x[t];  y_2w[t] = y_w[t] + y_w[t + w]   for 0 <= t <= N - 2w.
//   3. snr_w[t] = (double(y_w[t]) - w*mu) * r_w   with r_w = 1 / (sqrt(var) * sqrt(double(w))), IEEE double,
//      evaluated exactly in this order (built with -ffp-contract=off).
//   4. every (row, w, t) with snr_w[t] >= threshold is a candidate {dm_index, width, t, snr}; listed
//      here in (row, w, t) ascending order (the GPU lists them in any order).
//
// Pins (tests/test_oracle_pins.py): closed forms (alternating +-1 row; a lone width-w pulse on a zero row),
// brute-force numpy recomputation with direct (non-doubling) window sums on integer rows, constant rows.
//
// Build: g++ -O3 -std=c++17 -ffp-contract=off -fPIC -shared (oracle/__init__.py).
#include <cmath>
#include <cstdint>
#include <type_traits>
#include <vector>

namespace {

struct Cand { int32_t dm_index; int32_t width; int64_t t; double snr; };

template <typename T>
long long detect_rows(const T* x, long long stride, int nrows, long long n, int nwidths, double threshold,
                      Cand* out, long long max_out) {
    long long count = 0;
    std::vector<T> y((size_t)n), z((size_t)n);
    for (int r = 0; r < nrows; ++r) {
        const T* row = x + (long long)r * stride;
        double mu, var;
        if (std::is_integral<T>::value) {   // integer rows: exact sums
            int64_t s1 = 0, s2 = 0;
            for (long long t = 0; t < n; ++t) { s1 += (int64_t)row[t]; s2 += (int64_t)row[t] * (int64_t)row[t]; }
            mu = (double)s1 / (double)n;
            var = (double)s2 / (double)n - mu * mu;
        } else {
            double s1 = 0.0, s2 = 0.0;
            for (long long t = 0; t < n; ++t) { const double v = (double)row[t]; s1 += v; s2 += v * v; }
            mu = s1 / (double)n;
            var = s2 / (double)n - mu * mu;
        }
        if (!(var > 0.0)) continue;
        const double sd = std::sqrt(var);
        for (long long t = 0; t < n; ++t) y[(size_t)t] = row[t];
        long long w = 1;
        for (int k = 0; k < nwidths; ++k, w *= 2) {
            if (w > n) break;
            if (k > 0) {   // y_w[t] = y_{w/2}[t] + y_{w/2}[t + w/2]
                const long long h = w / 2;
                for (long long t = 0; t + w <= n; ++t) z[(size_t)t] = (T)(y[(size_t)t] + y[(size_t)(t + h)]);
                y.swap(z);
            }
            const double wm = (double)w * mu;
            const double rw = 1.0 / (sd * std::sqrt((double)w));
            for (long long t = 0; t + w <= n; ++t) {
                const double snr = ((double)y[(size_t)t] - wm) * rw;
                if (snr >= threshold) {
                    if (count < max_out) out[count] = Cand{r, (int32_t)w, t, snr};
                    ++count;
                }
            }
        }
    }
    return count;
}

}  // namespace

extern "C" {

// Returns the number of candidates (may exceed max_out: the first max_out are stored), or -1 on bad arguments.
long long oracle_detect_i32(const int32_t* x, long long stride, int nrows, long long n, int nwidths, double threshold,
                            void* out, long long max_out) {
    if (!x || nrows < 0 || n < 1 || nwidths < 1 || nwidths > 16 || stride < n || max_out < 0 || (max_out && !out)) return -1;
    return detect_rows<int32_t>(x, stride, nrows, n, nwidths, threshold, (Cand*)out, max_out);
}
long long oracle_detect_f32(const float* x, long long stride, int nrows, long long n, int nwidths, double threshold,
                            void* out, long long max_out) {
    if (!x || nrows < 0 || n < 1 || nwidths < 1 || nwidths > 16 || stride < n || max_out < 0 || (max_out && !out)) return -1;
    return detect_rows<float>(x, stride, nrows, n, nwidths, threshold, (Cand*)out, max_out);
}

}  // extern "C"
