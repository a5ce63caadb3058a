// plan.h — internal plan object of libdedisp_b200 (not part of the C ABI; see include/dedisp.h).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/dedisp.h"

// Geometry of the TILED kernel chosen at plan time (kernels_tiled.cuh).
struct TiledGeom {
    bool ok = false;
    int dt = 0;          // DM rows per thread; CTA covers 8*dt rows
    int slot_bytes = 0;  // shared-memory bytes reserved per staged channel window
    int cb = 0;          // channels per pipeline stage
};

// One pass of the SUBBAND kernel = one sub-band of channels [c_begin, c_end) (subband.h).
struct SubbandGeom {
    bool ok = false;
    int variant = 0;                 // index into the kernel variant table
    std::vector<int> first_chan;     // G+1 boundaries
    int ngroups = 0;                 // DM groups of SB_D rows
    int max_skew = 0;                // max over passes/CTAs of the parallelogram skew (samples)
    std::vector<uint32_t> win_len;   // per (pass, cta-row-block, channel) staged window length
    std::vector<uint64_t> records;   // packed per (channel, DM group) records, see subband.h
    std::vector<int32_t> cta_meta;   // per (channel, cta-row-block): window start rel. to skew origin
    uint64_t *d_records = nullptr;
    int32_t *d_cta_meta = nullptr;
    int32_t *d_skew = nullptr;       // per (pass, d): s(c_ref(pass), d)
    std::vector<int32_t> skew;
    int slot_words = 0;
    int cb = 0;
};

struct dedisp_plan {
    int nchans = 0, ndm = 0, dtype = 0;
    double fch1 = 0, foff = 0, tsamp = 0;
    unsigned flags = 0;
    std::vector<double> dm;
    std::vector<int32_t> shifts;  // [c][d]
    long long maxshift = 0;
    int32_t *d_shifts = nullptr;
    int kernel = DEDISP_KERNEL_AUTO;  // requested
    int device = -1;
    int sm_count = 0;
    TiledGeom tiled;
    SubbandGeom sb;
    std::string cuda_err;
    // scratch of dedisp_execute_host (grown on demand, freed at destroy)
    void *d_host_in = nullptr, *d_host_out = nullptr;
    size_t host_in_bytes = 0, host_out_bytes = 0;
};

inline int dtype_esize(int dtype) { return dtype == DEDISP_U8 ? 1 : dtype == DEDISP_F16 ? 2 : 4; }

// shift_table.cpp (host, IEEE double, compiled with -ffp-contract=off)
int build_shift_table(int nchans, double fch1, double foff, double tsamp, const double *dm, int ndm,
                      int32_t *table, long long *maxshift);

// Beam batching: one launch covers `n` independent beams (grid.z), beam b at d_in + b*in_stride
// and d_out + b*out_stride (strides in ELEMENTS).
struct Batch {
    int n = 1;
    long long in_stride = 0, out_stride = 0;
};

// kernels_tiled.cu
void tiled_choose_geom(dedisp_plan *p);
cudaError_t launch_naive(const dedisp_plan *p, const void *d_in, long long in_stride, long long nsamp_out,
                         void *d_out, long long out_stride, Batch b, cudaStream_t st);
cudaError_t launch_tiled(const dedisp_plan *p, const void *d_in, long long in_stride, long long nsamp_out,
                         void *d_out, long long out_stride, Batch b, cudaStream_t st);

// subband.cu
void subband_build(dedisp_plan *p);            // host tables; sets p->sb.ok
cudaError_t subband_upload(dedisp_plan *p);
void subband_free(dedisp_plan *p);
long long subband_verify_records(const dedisp_plan *p);
cudaError_t launch_subband(const dedisp_plan *p, const void *d_in, long long in_stride, long long nsamp_out,
                           void *d_out, long long out_stride, Batch b, cudaStream_t st);

// plan.cu (shared by the ABI entry points and stream.cu)
int execute_impl(dedisp_plan *p, const void *d_in, long long in_stride, long long nsamp_out, void *d_out,
                 long long out_stride, Batch b, cudaStream_t st);
