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

// SUBBAND kernel (subband.cu): exact sub-band re-skewed multi-pass with register-window reuse.
// Thread tile = SB_D DM rows x SB_K consecutive samples; warp = one DM group (SB_D rows) x 32 lanes;
// CTA = SB_WARPS groups x SB_T samples in the pass's skewed time coordinate u = t + s(c_ref, d).
// The channel loop is generated threaded code (gen_subband_rows.py -> subband_rows.inc): per channel
// one jump per group of SB_G rows on the group's joint offset pattern (window in 8-byte pairs, in-window
// offsets 0..SB_S+1).
#ifndef SB_D_CFG
#define SB_D_CFG 4
#define SB_G_CFG 2
#define SB_K_CFG 26
#endif
#ifndef SB_S_CFG
#define SB_S_CFG 5
#endif
#ifndef SB_WARPS_CFG
#define SB_WARPS_CFG 12
#endif
constexpr int SB_D = SB_D_CFG;
constexpr int SB_K = SB_K_CFG;
constexpr int SB_T = 32 * SB_K;       // u-samples per CTA tile
constexpr int SB_WARPS = SB_WARPS_CFG; // DM groups per CTA (one warp each)
constexpr int SB_ROWS = SB_D * SB_WARPS;
constexpr int SB_G = SB_G_CFG;        // rows per dispatch group
constexpr int SB_S = SB_S_CFG;        // largest spread of the residual delay over a thread's rows
constexpr int SB_OMAX = SB_S + 1;     // largest in-window offset a row may have
constexpr int SB_WPAIRS = (SB_K + SB_OMAX + 1) / 2;    // 8-byte pairs a thread loads per channel
constexpr int SB_REC_STRIDE = SB_WARPS * 8;            // bytes between a warp's records of consecutive staged channels
#ifndef SB_CB_CFG
#define SB_CB_CFG 8
#endif
constexpr int SB_CB = SB_CB_CFG;      // smallest number of channels per pipeline stage (one staging warp each)
#ifndef SB_STAGES_CFG
#define SB_STAGES_CFG 2
#endif
constexpr int SB_STAGES = SB_STAGES_CFG;
#ifndef SB_CB_MAX_CFG
#define SB_CB_MAX_CFG 16
#endif
constexpr int SB_CB_MAX = SB_CB_MAX_CFG;  // channels per stage are chosen at plan build (as many as fit, at most this)
constexpr int SB_EP_WORDS = SB_T + 8;     // epilogue transpose buffer of one warp: one row of the tile, shifted by up to 3 words
// staged 16-byte chunks per channel the slot can hold, a multiple of 32
constexpr int SB_NCH_MAX = ((SB_K * 31 + 2 * SB_WPAIRS + 3) / 4 + 96 + 31) / 32 * 32;

// Packed 16-bit variant for u8 plans (subband_rows_i16.inc): a 32-bit word holds TWO samples, so the same
// thread tile of SB_K words covers 2*SB_K samples per row, and the sums run on the integer pipes
// (profiles/r2_microbench.md, packed_add.cu). Offsets are in samples; window bases stay 8 bytes = 4 samples apart.
constexpr int SB16_KS = 2 * SB_K;         // samples per thread and row
constexpr int SB16_T = 32 * SB16_KS;      // u-samples per CTA tile
#ifndef SB16_OMAX_CFG
#define SB16_OMAX_CFG 11
#endif
constexpr int SB16_OMAX = SB16_OMAX_CFG;  // largest in-window offset (11: word offset 5 + the half-word bit)
constexpr int SB16_S = SB16_OMAX - 3;     // spread bound of a thread's rows (the smallest offset is 0..3)
constexpr int SB16_CHMAX = 257;           // channels per pass: 257 * 255 = 65535 still fits a 16-bit lane
constexpr int SB16_EP_WORDS = SB16_T + 8;
constexpr int SB16_WPAIRS = ((SB16_OMAX >> 1) + SB_K + 2) / 2;   // 8-byte pairs a thread loads per channel (its own count: the fp32 loop's may differ)

struct SubbandPass {
    int c_begin = 0, c_end = 0, c_ref = 0;
    int max_skew = 0;                 // max over the pass's DM rows of s(c_ref, d)
    int blk_begin = 0, blk_end = 0;   // DM blocks this pass covers (a plan may cut its DM blocks into ranges)
    bool first = false;               // first pass of its DM range: stores instead of adding
};

// device copy of a pass (the kernel walks a range of these; nothing in it depends on nsamp_out)
struct SbPassDev {
    int c_begin, c_end;
    int blk_begin, blk_end;
    int max_skew;
    int first;
    int pad0, pad1;                   // pad0: 1 = last sub-band of its DM range (stores when the launches run in reverse order)
};

// What one SUBBAND launch sequence covers: launch-order range of passes, DM-block range, order, and
// (dedisp_execute_host) one "rows of pass g are on the device" event per pass. Passed by the caller;
// the plan itself stays read-only during execute.
struct SbRun {
    int pass_lo = 0, pass_hi = -1;     // launch-order indices (-1: all)
    int blk_lo = 0, blk_hi = -1;       // DM blocks (-1: all)
    bool reverse = false;              // run the passes last sub-band first
    const cudaEvent_t *pass_ready = nullptr;
    int tm_bits = 0;                   // != 0: d_in is TIME-major, tm_bits (1/2/4/8) per sample, in_stride = bytes per time sample
};

struct SubbandGeom {
    bool ok = false;
    bool i16 = false;                 // u8 plan summed as packed 16-bit pairs (units below in samples all the same)
    int tile_t = SB_T;                // u-samples per CTA tile (SB_T or SB16_T)
    std::vector<SubbandPass> passes;  // launch order: the k-th sub-band of every DM range, k = 0, 1, ...
    std::vector<int> launch_begin;    // [nlaunch + 1]: ordered launch g runs passes [launch_begin[g], launch_begin[g + 1])
    int ngroups = 0, nblk = 0;
    int nranges = 0;                  // DM-block ranges, each with its own sub-band partition (1 for uniform DM plans)
    // [nblk][nchans][SB_WARPS] per (block, channel, group): low word = joint pattern ids, 8 bits per dispatch group (group 0 lowest):
    // (o_a*(S+2) + o_b)... (i16: one offset per row, 8 bits each, row 0 lowest), high word = window base a in 8-byte pairs (subband.cu)
    std::vector<uint64_t> records;
    // per (block, channel): {window base r (multiple of 4 samples, i16: 8; relative to u), 16-byte chunks to stage}
    std::vector<int32_t> meta;        // [nblk][nchans][2]
    std::vector<int32_t> skew;        // [npasses][ndm] = s(c_ref(pass), d)
    uint64_t *d_records = nullptr;
    int32_t *d_meta = nullptr;
    int32_t *d_skew = nullptr;
    SbPassDev *d_passes = nullptr;    // [npasses]
    int max_nch = 0;                  // largest staged chunk count (sizes the shared-memory slot)
    int slot_chunks = 0, cb = 0;      // launch geometry fixed at upload: slot size, channels per stage
    size_t smem = 0;                  // dynamic shared memory of the kernel
    int raw_slot_bytes = 0, cb_raw = 0;   // the same for the raw path (u8 / f16 input, unaligned fp32 rows)
    size_t smem_raw = 0;
};

struct dedisp_plan {
    int nchans = 0, ndm = 0, dtype = 0;
    double fch1 = 0, foff = 0, tsamp = 0;
    unsigned flags = 0;
    bool time_major = false;          // DEDISP_PLAN_TIME_MAJOR: sub-bands cut at multiples of 16 channels
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
    // dedisp_execute_host overlap: a copy stream and one "rows of pass g are on the device" event per pass
    cudaStream_t host_copy_st = nullptr;
    std::vector<cudaEvent_t> host_pass_ready;
    bool merge_fp_passes = false;             // fp plans: run all passes in one launch (sums not bit-reproducible)
    cudaStream_t host_d2h_st = nullptr;
    std::vector<cudaEvent_t> host_slab_done;
    int host_slabs = 0;                       // DM slabs the last dedisp_execute_host call ran its last pass in (0: no slab overlap)
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
int subband_launches(const dedisp_plan *p, int resolved_kernel);  // kernel launches per execute
bool subband_smem_fits(const dedisp_plan *p);
bool subband_merges(const dedisp_plan *p);      // all passes of an execute in one launch?
cudaError_t launch_subband(dedisp_plan *p, const void *d_in, long long in_stride, long long nsamp_out,
                           void *d_out, long long out_stride, Batch b, cudaStream_t st, const SbRun &run);

// plan.cu (shared by the ABI entry points and stream.cu)
int execute_impl(dedisp_plan *p, const void *d_in, long long in_stride, long long nsamp_out, void *d_out,
                 long long out_stride, Batch b, cudaStream_t st, const SbRun &run = SbRun());
