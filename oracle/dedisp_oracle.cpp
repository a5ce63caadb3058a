// ORACLE — test infrastructure, NOT the product.
//
// Plain, slow, single-threaded CPU statement of brute-force incoherent
// de-dispersion, written from the paper's definition. Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may load this library. It shares no code (no header, no helper, no table
// generator) with paper_1111_6399_b200/csrc/.
//
// What it computes (§2: "shifting each frequency channel by the
// appropriate amount of time for each DM being searched" ... "before frequency
// integration"; formula fixed by BASELINE.json:north_star):
//
//     out[d][t] = sum_{c=0}^{nchans-1} in[c][ t + s(c,d) ]
//     s(c,d)    = floor( 4.148808e3 * DM_d * (f_c^-2 - f_top^-2) / tsamp + 0.5 )
//
// f in MHz, tsamp in s, f_c = fch1 + c*foff, f_top = fch1 (DESIGN.md readings
// R1-R5). Input is channel-major, time contiguous (Fig. 2 caption:
// "cache-lines of constant frequency, contiguous time").
//
// Pins (tests/test_oracle_pins.py): DM=0 row == plain channel sum; unit-impulse
// response; noise-free pulse peak == nchans*amp; per-(d,t) brute force on tiny
// inputs with the delay recomputed inline; textbook delay in ms/GHz form;
// shift-table regression values (tests/golden/shift_pins.txt).
//
// Build: g++ -O3 -std=c++17 -ffp-contract=off -fPIC -shared (see oracle/build.py).

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

// Step 2 of SURVEY.md §8(c): the normative expression, IEEE double, this order.
long long delay_samples(double fch1, double foff, double tsamp, double dm, int c) {
    const double f_c = fch1 + (double)c * foff;
    const double f_top = fch1;
    const double x = ((4.148808e3 * dm) * (1.0 / (f_c * f_c) - 1.0 / (f_top * f_top))) / tsamp;
    return (long long)std::floor(x + 0.5);
}

// IEEE-754 binary16 bit pattern -> double, exact.
double half_bits_to_double(uint16_t h) {
    const int sign = (h >> 15) & 1;
    const int expo = (h >> 10) & 0x1f;
    const int frac = h & 0x3ff;
    double v;
    if (expo == 0) {
        v = std::ldexp((double)frac, -24);            // subnormal: frac * 2^-24
    } else if (expo == 31) {
        v = frac ? NAN : INFINITY;
    } else {
        v = std::ldexp((double)(frac | 0x400), expo - 25);  // (1.frac) * 2^(expo-15)
    }
    return sign ? -v : v;
}

struct F32Elem { static double get(const void* p, long long i) { return (double)((const float*)p)[i]; } };
struct F16Elem { static double get(const void* p, long long i) { return half_bits_to_double(((const uint16_t*)p)[i]); } };

// Step 4: for d: for c: for t. Double accumulator. abs_sum is the tolerance
// denominator sum_c |in[c][t+s]| (north_star: "max relative error 1e-5 of the
// sum of |terms|").
template <class Elem>
int dedisperse_fp(int nchans, double fch1, double foff, double tsamp,
                  const double* dm_list, const int* dm_rows, int nrows,
                  const void* in, long long in_stride, long long nsamp_in, long long nsamp_out,
                  double* out, double* abs_sum) {
    if (nchans < 1 || nrows < 0 || nsamp_out < 1 || !in || !out) return 1;
    std::vector<double> acc((size_t)nsamp_out), aacc((size_t)nsamp_out);
    for (int r = 0; r < nrows; ++r) {
        const double dm = dm_list[dm_rows[r]];
        for (long long t = 0; t < nsamp_out; ++t) { acc[t] = 0.0; aacc[t] = 0.0; }
        for (int c = 0; c < nchans; ++c) {
            const long long s = delay_samples(fch1, foff, tsamp, dm, c);
            if (s < 0 || s + nsamp_out > nsamp_in) return 2;      // no padding, no wrap (reading R10)
            const long long base = (long long)c * in_stride + s;
            for (long long t = 0; t < nsamp_out; ++t) {
                const double v = Elem::get(in, base + t);
                acc[t] += v;
                aacc[t] += std::fabs(v);
            }
        }
        std::memcpy(out + (size_t)r * nsamp_out, acc.data(), sizeof(double) * (size_t)nsamp_out);
        if (abs_sum) std::memcpy(abs_sum + (size_t)r * nsamp_out, aacc.data(), sizeof(double) * (size_t)nsamp_out);
    }
    return 0;
}

}  // namespace

extern "C" {

// s(c,d) for every (c,d): table[c*ndm + d]. Returns 0.
int oracle_shift_table(int nchans, double fch1, double foff, double tsamp,
                       const double* dm_list, int ndm, long long* table) {
    if (nchans < 1 || ndm < 1 || !dm_list || !table) return 1;
    for (int c = 0; c < nchans; ++c)
        for (int d = 0; d < ndm; ++d)
            table[(size_t)c * ndm + d] = delay_samples(fch1, foff, tsamp, dm_list[d], c);
    return 0;
}

// Step 3: maxshift = max over (c,d) of s(c,d).
long long oracle_max_shift(int nchans, double fch1, double foff, double tsamp,
                           const double* dm_list, int ndm) {
    long long m = 0;
    for (int c = 0; c < nchans; ++c)
        for (int d = 0; d < ndm; ++d) {
            const long long s = delay_samples(fch1, foff, tsamp, dm_list[d], c);
            if (s > m) m = s;
        }
    return m;
}

// U8 input: int64 accumulate, checked to fit int32, stored int32 (step 4).
// Computes rows dm_rows[0..nrows) of the plan; out is [nrows][nsamp_out].
// Return: 0 ok, 1 bad args, 2 shift leaves the input, 3 int32 overflow.
int oracle_dedisperse_u8(int nchans, double fch1, double foff, double tsamp,
                         const double* dm_list, const int* dm_rows, int nrows,
                         const uint8_t* in, long long in_stride, long long nsamp_in,
                         long long nsamp_out, int32_t* out) {
    if (nchans < 1 || nrows < 0 || nsamp_out < 1 || !in || !out) return 1;
    std::vector<int64_t> acc((size_t)nsamp_out);
    for (int r = 0; r < nrows; ++r) {
        const double dm = dm_list[dm_rows[r]];
        for (long long t = 0; t < nsamp_out; ++t) acc[t] = 0;
        for (int c = 0; c < nchans; ++c) {
            const long long s = delay_samples(fch1, foff, tsamp, dm, c);
            if (s < 0 || s + nsamp_out > nsamp_in) return 2;
            const uint8_t* row = in + (long long)c * in_stride + s;
            for (long long t = 0; t < nsamp_out; ++t) acc[t] += row[t];
        }
        for (long long t = 0; t < nsamp_out; ++t) {
            if (acc[t] > INT32_MAX) return 3;
            out[(size_t)r * nsamp_out + t] = (int32_t)acc[t];
        }
    }
    return 0;
}

int oracle_dedisperse_f32(int nchans, double fch1, double foff, double tsamp,
                          const double* dm_list, const int* dm_rows, int nrows,
                          const float* in, long long in_stride, long long nsamp_in,
                          long long nsamp_out, double* out, double* abs_sum) {
    return dedisperse_fp<F32Elem>(nchans, fch1, foff, tsamp, dm_list, dm_rows, nrows,
                                  in, in_stride, nsamp_in, nsamp_out, out, abs_sum);
}

// in: IEEE binary16 bit patterns.
int oracle_dedisperse_f16(int nchans, double fch1, double foff, double tsamp,
                          const double* dm_list, const int* dm_rows, int nrows,
                          const uint16_t* in, long long in_stride, long long nsamp_in,
                          long long nsamp_out, double* out, double* abs_sum) {
    return dedisperse_fp<F16Elem>(nchans, fch1, foff, tsamp, dm_list, dm_rows, nrows,
                                  in, in_stride, nsamp_in, nsamp_out, out, abs_sum);
}

// Step 5 (diagnostic only, not the acceptance test): float accumulator,
// channels in ascending order.
int oracle_dedisperse_f32_seq(int nchans, double fch1, double foff, double tsamp,
                              const double* dm_list, const int* dm_rows, int nrows,
                              const float* in, long long in_stride, long long nsamp_in,
                              long long nsamp_out, float* out) {
    if (nchans < 1 || nrows < 0 || nsamp_out < 1 || !in || !out) return 1;
    for (int r = 0; r < nrows; ++r) {
        const double dm = dm_list[dm_rows[r]];
        float* acc = out + (size_t)r * nsamp_out;
        for (long long t = 0; t < nsamp_out; ++t) acc[t] = 0.0f;
        for (int c = 0; c < nchans; ++c) {
            const long long s = delay_samples(fch1, foff, tsamp, dm, c);
            if (s < 0 || s + nsamp_out > nsamp_in) return 2;
            const float* row = in + (long long)c * in_stride + s;
            for (long long t = 0; t < nsamp_out; ++t) acc[t] = acc[t] + row[t];
        }
    }
    return 0;
}

}  // extern "C"
