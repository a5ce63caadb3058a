// ORACLE — test infrastructure, NOT the product.
//
// Plain CPU statement of the step in front of the de-dispersion hot path (
// PAPER.md:26 §1 names the stage chain "... integration, real-time dispersion searches"
// Fig. 2 caption fixes what the de-dispersion kernel wants: "cache-lines of constant frequency,
// contiguous time"): telescope back-ends deliver TIME-major data, one row per time sample holding all
// channels, usually packed to 1, 2, 4 or 8 bits per sample. This file unpacks and corner-turns such a
// block into the channel-major uint8 array that oracle/dedisp_oracle.cpp consumes. It shares no code
// with paper_1111_6399_b200/csrc/ and nothing with dedisp_oracle.cpp either.
//
// Layout (reading R15; the paper gives none): sample (t, c) is the nbits-wide unsigned
// integer in bits [ (c*nbits) mod 8, (c*nbits) mod 8 + nbits ) of byte (c*nbits)/8 of row t, i.e. the
// first channel sits in the LEAST significant bits of a byte (the sigproc filterbank convention).
// Rows are row_bytes apart (>= ceil(nchans*nbits/8)).
//
// Pins (tests/test_oracle_pins.py): hand-packed bytes for every nbits; numpy's independent
// unpackbits(bitorder="little") on random rows; pack -> unpack round trip; nbits = 8 is a transpose.
//
// Build: g++ -O3 -std=c++17 -fPIC -shared (oracle/__init__.py).
#include <cstdint>

extern "C" {

// out[c*out_stride + t] = sample (t, c), for 0 <= t < nsamp, 0 <= c < nchans. Returns 0, or 1 on bad
// arguments (nbits not in {1,2,4,8}, row too short, NULLs).
int oracle_unpack_time_major(const uint8_t* in, long long row_bytes, long long nsamp, int nchans, int nbits,
                             uint8_t* out, long long out_stride) {
    if (!in || !out || nsamp < 0 || nchans < 1) return 1;
    if (nbits != 1 && nbits != 2 && nbits != 4 && nbits != 8) return 1;
    if (row_bytes * 8 < (long long)nchans * nbits || out_stride < nsamp) return 1;
    const unsigned mask = (1u << nbits) - 1u;
    for (long long t = 0; t < nsamp; ++t) {
        const uint8_t* row = in + t * row_bytes;
        for (int c = 0; c < nchans; ++c) {
            const long long bit = (long long)c * nbits;
            out[(long long)c * out_stride + t] = (uint8_t)((row[bit / 8] >> (bit % 8)) & mask);
        }
    }
    return 0;
}

}  // extern "C"
