/* dedisp.h — C ABI of libdedisp_b200: brute-force incoherent de-dispersion on one B200 (sm_100a).
 *
 * The operation (§2: "shifting each frequency channel by the appropriate amount of
 * time for each DM being searched" ... "before frequency integration"; formula fixed by
 * BASELINE.json:north_star, readings R1-R10 in DESIGN.md):
 *
 *     out[d][t] = sum_{c=0}^{nchans-1} in[c][ t + s(c,d) ]        0 <= d < ndm, 0 <= t < nsamp_out
 *     s(c,d)    = floor( 4.148808e3 * DM_d * (f_c^-2 - f_top^-2) / tsamp + 0.5 )
 *
 * evaluated in IEEE double on the host; f_c = fch1 + c*foff (MHz, foff < 0), f_top = fch1,
 * tsamp in seconds. Input is channel-major with time contiguous (Fig. 2 caption:
 * "cache-lines of constant frequency, contiguous time"). Every (d,c,t) term is added — the
 * method is brute force, nothing is approximated or shared between trials.
 *
 * Conventions for every entry point:
 *   - returns a dedisp_status; no exception or abort crosses the ABI;
 *   - pointers named h_* are HOST memory, d_* are DEVICE memory of the current CUDA device;
 *   - the caller owns every buffer it passes in; the plan owns its own host and device tables;
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream);
 *   - there is no CPU fallback: on a machine without an sm_100 GPU plan creation fails with
 *     DEDISP_EUNSUPPORTED / DEDISP_ECUDA (except DEDISP_PLAN_HOST_ONLY plans, which can only be
 *     inspected, never executed).
 */
#ifndef DEDISP_B200_H
#define DEDISP_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dedisp_plan dedisp_plan;     /* opaque */
typedef struct dedisp_stream dedisp_stream; /* opaque: streaming multi-beam driver */

enum dedisp_dtype { DEDISP_U8 = 0, DEDISP_F16 = 1, DEDISP_F32 = 2 };

enum dedisp_status {
    DEDISP_OK = 0,
    DEDISP_EINVAL = 1,       /* bad argument (see each call) */
    DEDISP_ENOMEM = 2,       /* host or device allocation failed */
    DEDISP_ECUDA = 3,        /* a CUDA call failed; text via dedisp_last_cuda_error */
    DEDISP_EUNSUPPORTED = 4, /* device is not sm_100, or maxshift >= 2^31, or plan is host-only */
    DEDISP_ETOOLARGE = 5     /* a size exceeds the fixed scratch of a no-allocation entry point (dedisp_detect_static) */
};

/* Kernel selection (dedisp_plan_set_kernel). AUTO picks SUBBAND when the plan admits it and its passes
 * are not too short (about 20 channels per pass on average), else TILED, else NAIVE.
 * NAIVE is the one-thread-per-(d,t) cross-check kernel used by the parity tests' chain of trust. */
enum dedisp_kernel {
    DEDISP_KERNEL_AUTO = 0,
    DEDISP_KERNEL_NAIVE = 1,   /* global loads through L1, no staging */
    DEDISP_KERNEL_TILED = 2,   /* CTA = DM tile x time tile, channel windows staged in shared memory */
    DEDISP_KERNEL_SUBBAND = 3  /* exact sub-band re-skewed multi-pass with register-window reuse */
};

enum dedisp_plan_flags {
    DEDISP_PLAN_DEFAULT = 0,
    DEDISP_PLAN_HOST_ONLY = 1, /* build host tables only; no CUDA call is made; execute -> EUNSUPPORTED */
    DEDISP_PLAN_TIME_MAJOR = 2, /* the plan will be fed TIME-major packed input through dedisp_execute_time_major:
                                  in_dtype must be DEDISP_U8 and nchans a multiple of 16 (else EINVAL); sub-bands
                                  are cut at multiples of 16 channels. Channel-major calls stay available. */
    DEDISP_PLAN_NO_PACKED = 4  /* DEDISP_U8 plans: sum in fp32 like the other dtypes instead of as packed 16-bit
                                  pairs on the integer pipes (same results bit for bit; kept for comparison) */
};

/* ---- subsystem (2): shift-table builder ("the shifting value
 * is calculated using as few operations as possible" — here: once per plan, on the host, in double).
 *
 * dedisp_shift_table_host: pure host function, no CUDA. Writes s(c,d) to h_table[c*ndm + d]
 * (int32) and the maximum to *h_maxshift (may be NULL). EINVAL on nchans<1, ndm<1, tsamp<=0,
 * fch1<=0, foff>=0, lowest channel frequency <=0, DM negative / non-finite / decreasing, NULLs;
 * EUNSUPPORTED if any shift >= 2^31. */
int dedisp_shift_table_host(int nchans, double fch1_mhz, double foff_mhz, double tsamp_s,
                            const double *h_dm_list, int ndm, int *h_table, long long *h_maxshift);

/* ---- subsystem (1): plan / execute / destroy (BASELINE.json:north_star (1)).
 *
 * dedisp_plan_create: validates (same rules as dedisp_shift_table_host, plus in_dtype), builds the
 * shift table and the kernels' tiling/sub-band metadata on the host, uploads them to the current
 * device. h_dm_list[ndm] is copied. in_dtype is a dedisp_dtype. */
int dedisp_plan_create(dedisp_plan **plan, int nchans, double fch1_mhz, double foff_mhz,
                       double tsamp_s, const double *h_dm_list, int ndm, int in_dtype);
int dedisp_plan_create_ex(dedisp_plan **plan, int nchans, double fch1_mhz, double foff_mhz,
                          double tsamp_s, const double *h_dm_list, int ndm, int in_dtype,
                          unsigned flags);

/* dedisp_execute: out[d][t] for all ndm trials and 0 <= t < nsamp_out, asynchronously on `stream`.
 *   d_in : [nchans][nsamp_out + maxshift] elements of in_dtype, dense rows (row stride =
 *          nsamp_out + dedisp_plan_max_shift(plan)); channel 0 = fch1 (highest frequency).
 *   d_out: [ndm][nsamp_out], row stride nsamp_out; int32 for DEDISP_U8 input (exact), float32 for
 *          DEDISP_F16 / DEDISP_F32 input (fp32 accumulation; summation order unspecified).
 * May be called repeatedly. The call allocates nothing, does not synchronise, and leaves the plan
 * read-only for every input dtype, so calls on one plan may run concurrently on different streams.
 * (u8 / f16 input and fp32 rows that are not 16-byte aligned are converted / realigned inside the
 * SUBBAND kernel's staging step; there is no scratch copy of the input.) EINVAL: NULLs, nsamp_out < 1. */
int dedisp_execute(dedisp_plan *plan, const void *d_in, long long nsamp_out, void *d_out,
                   void *stream);

/* Fused corner turn + unpack (the stage in front of the
 * "real-time dispersion searches" delivers time-major data; the kernel wants "cache-lines of
 * constant frequency, contiguous time"). d_in is TIME-major (sigproc filterbank order): row t, 0 <= t <
 * nsamp_out + maxshift, holds all channels of time sample t as nbits-wide unsigned integers, nbits in
 * {1, 2, 4, 8}; sample (t, c) occupies bits [(c*nbits) mod 8, +nbits) of byte (c*nbits)/8 of the row (first
 * channel in the least significant bits). Rows are row_bytes apart. The SUBBAND kernel's producer warps
 * read these rows directly and write fp32 channel windows into the pipeline ring: no transposed or
 * unpacked copy of the input exists in HBM. d_out: [ndm][nsamp_out] int32, exact.
 * The plan must have been created with DEDISP_PLAN_TIME_MAJOR and admit the SUBBAND kernel
 * (EUNSUPPORTED otherwise). EINVAL: NULLs, nbits not in {1,2,4,8}, row_bytes < nchans*nbits/8, d_in or
 * row_bytes not 16-byte aligned. Allocates nothing; asynchronous on `stream`. */
int dedisp_execute_time_major(dedisp_plan *plan, const void *d_in, int nbits, long long row_bytes,
                              long long nsamp_out, void *d_out, void *stream);

/* Same with explicit row strides in ELEMENTS (in_stride >= nsamp_out + maxshift, out_stride >=
 * nsamp_out), else EINVAL. Any base address and any stride are correct; a 16-byte-aligned d_in and
 * in_stride*elemsize let fp32 input take the direct TMA path, a 16-byte-aligned d_out and
 * out_stride*4 let the epilogue use vector stores / reductions. The TILED kernel, when forced with
 * dedisp_plan_set_kernel, requires a 16-byte-aligned d_in (EINVAL otherwise); AUTO never fails on
 * alignment. */
int dedisp_execute_strided(dedisp_plan *plan, const void *d_in, long long in_stride_elems,
                           long long nsamp_out, void *d_out, long long out_stride_elems,
                           void *stream);

/* Beam batching (north_star (4) "batches beams"): nbeams independent inputs through one plan in one
 * launch. Beam b reads d_in + b*in_beam_stride_elems and writes d_out + b*out_beam_stride_elems
 * (ELEMENTS of the input / output type); each beam is laid out as in dedisp_execute_strided.
 * EINVAL: nbeams < 1 or > 65535, beam strides smaller than one beam's extent. */
int dedisp_execute_batched(dedisp_plan *plan, int nbeams, const void *d_in, long long in_stride_elems,
                           long long in_beam_stride_elems, long long nsamp_out, void *d_out,
                           long long out_stride_elems, long long out_beam_stride_elems, void *stream);

/* Host-buffer convenience (the end-to-end call bench.py's "e2e" times): h_in [nchans][nsamp_out +
 * maxshift] and h_out [ndm][nsamp_out] are HOST buffers (pinned memory makes the copies
 * asynchronous to the host and full speed). Copies the input to plan-owned device scratch (grown
 * on demand, freed at destroy), executes, copies the result back and SYNCHRONISES `stream` before
 * returning. For the SUBBAND kernel with more than one launch (any in_dtype) the input is copied in the
 * order the launches need it (they run last sub-band first, so a growing suffix of the channels) on a
 * plan-owned second stream, ordered after `stream`, and the result per DM slab of the last two launches on
 * a third, so both transfers overlap the launches. Not re-entrant per plan (the scratch is shared). */
int dedisp_execute_host(dedisp_plan *plan, const void *h_in, long long nsamp_out, void *h_out,
                        void *stream);

int dedisp_plan_destroy(dedisp_plan *plan); /* NULL is OK */

/* ---- inspection */
long long dedisp_plan_max_shift(const dedisp_plan *plan); /* nsamp_in = nsamp_out + this; -1 on NULL */
int dedisp_plan_nchans(const dedisp_plan *plan);
int dedisp_plan_ndm(const dedisp_plan *plan);
/* Copies the plan's table to h_out[nchans*ndm] (index c*ndm + d). For the table-parity test. */
int dedisp_plan_get_shifts(const dedisp_plan *plan, int *h_out);
/* Force a kernel (enum dedisp_kernel). EUNSUPPORTED if the plan does not admit it. */
int dedisp_plan_set_kernel(dedisp_plan *plan, int kernel);
/* SUBBAND pass merging. The SUBBAND kernel runs one launch per sub-band pass, each adding its partial
 * sums into out in a fixed order (bit-reproducible results). With merging ON all passes run in ONE
 * launch: out is zeroed and every pass adds with L2 reductions in whatever order the hardware
 * schedules them. Integer-valued sums (DEDISP_U8 plans) are exact and therefore identical either way, so
 * u8 plans merge on their own whenever it is faster (many short passes); for DEDISP_F16 / DEDISP_F32
 * plans merging is OFF unless enabled here, and when ON the fp32 sums may differ in their last bits from run to run (still within the 1e-5 * sum|terms|
 * bound). on = 0 / 1; EINVAL on NULL. */
int dedisp_plan_set_pass_merge(dedisp_plan *plan, int on);
/* The kernel dedisp_execute will launch for this plan (resolved, never AUTO). */
int dedisp_plan_get_kernel(const dedisp_plan *plan);
/* Sub-band layout of the SUBBAND kernel: number of sub-bands G (0 if the plan has none) and, if
 * h_first_chan != NULL, the G+1 channel boundaries. A plan whose DM step changes (e.g. 0.1 / 0.25 /
 * 0.5) cuts its DM rows into ranges with one partition each; these two calls describe the first
 * range, dedisp_plan_launches_per_execute counts the launches of all of them. */
int dedisp_plan_num_subbands(const dedisp_plan *plan);
int dedisp_plan_get_subbands(const dedisp_plan *plan, int *h_first_chan /* [G+1] */);
/* Host check used by the CPU tests: rebuild s(c,d) for every (c,d) from the SUBBAND kernel's packed
 * per-(pass, DM group, channel) records and compare with the shift table. Returns the number of
 * mismatching entries (0 = the records encode exactly the table), or -1 if the plan has none. */
long long dedisp_plan_verify_records(const dedisp_plan *plan);
/* Number of kernel launches one dedisp_execute issues for this plan (for bench.py's gpu_launches). */
int dedisp_plan_launches_per_execute(const dedisp_plan *plan);

/* Launch geometry of the SUBBAND kernel for this plan, for reports: h_out[8] = {channels per pipeline
 * stage (aligned fp32 rows), the same for the raw path (u8 / f16 / unaligned rows), bytes per staged
 * channel window, dynamic shared memory of the two paths, DM blocks, DM ranges, passes}. Zeros if the
 * plan does not admit SUBBAND. */
int dedisp_plan_get_geometry(const dedisp_plan *plan, int *h_out);
/* Number of DM slabs the last dedisp_execute_host call on this plan ran its final pass(es) in (0: the
 * call did not take the slab-overlap path; else min(8, DM blocks)). For the tests that must know which path they exercised. */
int dedisp_plan_last_host_slabs(const dedisp_plan *plan);

/* ---- detection behind the hot path ("detect millisecond radio
 * bursts ... in real-time", "detection of interesting signals"). The paper gives no algorithm;
 * this is the build's own definition (reading R16), stated so that it can be checked exactly:
 * for every row x[0..nsamp) of a de-dispersed block d_block[ndm][stride] (int32 if block_is_float == 0,
 * else float32):
 *   1. S1 = sum x, S2 = sum x^2 (exact 64-bit integers for int32 rows, double for float rows), mu = S1/nsamp,
 *      var = S2/nsamp - mu*mu; rows with var <= 0 yield nothing;
 *   2. boxcar sums of width w = 1, 2, 4, ..., 2^(nwidths-1) by doubling in the row's own arithmetic:
 *      y_1 = x, y_2w[t] = y_w[t] + y_w[t + w], for windows that lie inside the row;
 *   3. snr_w[t] = (double(y_w[t]) - w*mu) * (1 / (sqrt(var) * sqrt(w))), IEEE double, each operation rounded
 *      (no contraction) - integer rows therefore give bit-identical values on any conforming machine;
 *   4. every (row, w, t) with snr_w[t] >= threshold is appended, in no particular order, to d_cands (device,
 *      capacity max_cands records; further ones are counted but not stored).
 * d_work: device scratch of dedisp_detect_workspace_bytes(ndm) bytes, 8-byte aligned, owned by the caller;
 * when the call's work on `stream` has completed its first 8 bytes hold the total number of candidates
 * (unsigned 64-bit). Allocates nothing, asynchronous on `stream`. EINVAL: NULLs, ndm < 1 or > 65535,
 * nsamp < 1, stride < nsamp, nwidths < 1 or > DEDISP_DETECT_MAX_WIDTHS. */
#define DEDISP_DETECT_MAX_WIDTHS 8
typedef struct dedisp_candidate {
    int dm_index;     /* row of the block */
    int width;        /* boxcar width w in samples */
    long long t;      /* first sample of the window */
    double snr;
} dedisp_candidate;
long long dedisp_detect_workspace_bytes(int ndm);
int dedisp_detect(const void *d_block, int block_is_float, int ndm, long long nsamp, long long stride, int nwidths,
                  double threshold, dedisp_candidate *d_cands, long long max_cands, void *d_work, void *stream);

/* dedisp_detect_static: dedisp_detect for callers that cannot call cudaMalloc and have no scratch buffer to hand
 * over (code under CUDA graph capture, tight serving loops, harnesses that forbid allocation). Same definition,
 * same kernels, same results as dedisp_detect; the per-row scratch ({S1, S2}, 16 bytes per DM row) lives in a
 * file-scope `static __device__` array inside the library: DEDISP_DETECT_STATIC_MAX_NDM rows = 128 KB, which
 * every GPU that loads the library holds until the process exits. The caller still owns inputs and outputs:
 * d_block and d_cands as for dedisp_detect, and d_count (device, 8-byte aligned, 8 bytes), which holds the total
 * number of candidates once the call's work on `stream` has completed.
 * Calls no cudaMalloc / cudaFree / allocating library routine: two cudaMemsetAsync (the scratch rows of this
 * call and *d_count start at zero; the array otherwise keeps the previous call's contents) and two kernel
 * launches on `stream`. The first call on each device also looks the array's device address up
 * (cudaGetSymbolAddress, with that device current; later calls reuse it), so make one call outside a graph
 * capture first.
 * ALL calls on a device share the one array: calls that overlap on the GPU (different streams, or different
 * threads or processes' streams of one context) race and give wrong statistics; serialise them on one stream
 * or with events, or use dedisp_detect with one workspace per stream.
 * ETOOLARGE: ndm > DEDISP_DETECT_STATIC_MAX_NDM (nothing is launched). EINVAL: as dedisp_detect, or d_count
 * NULL / misaligned. ECUDA: a CUDA call failed. */
#define DEDISP_DETECT_STATIC_MAX_NDM 8192
int dedisp_detect_static(const void *d_block, int block_is_float, int ndm, long long nsamp, long long stride, int nwidths,
                         double threshold, dedisp_candidate *d_cands, long long max_cands, unsigned long long *d_count,
                         void *stream);

const char *dedisp_error_string(int code);
const char *dedisp_last_cuda_error(const dedisp_plan *plan);

/* ---- subsystem (4): streaming multi-beam driver (the paper's MDSM
 * wrapper). Input chunk k holds samples [k*N, (k+1)*N) of every (beam, channel);
 * output block k holds out[.][t] for global t in [k*N - maxshift, (k+1)*N - maxshift): the history
 * before the first chunk is zero, so the first maxshift outputs of block 0 are warm-up.
 * Equivalent to one dedisp_execute over the whole stream delayed by maxshift.
 *
 * dedisp_stream_create: device buffers for nbeams x nchans x (maxshift + chunk) input (nbuffers
 * copies, >= 2, for copy/compute overlap) and nbeams x ndm x chunk output per buffer; one copy
 * stream, one compute stream. The plan must outlive the stream object. */
int dedisp_stream_create(dedisp_stream **s, dedisp_plan *plan, int nbeams, long long chunk_nsamp,
                         int nbuffers);
/* dedisp_stream_push: enqueue one chunk. h_chunk: host memory (pinned for true async copies),
 * layout [beam][chan][chunk_nsamp] of the plan's in_dtype. Returns immediately; *d_out (device,
 * [beam][ndm][chunk_nsamp], owned by the stream object, reused after nbuffers pushes) is valid
 * once *done_event (a cudaEvent_t as void*) has completed or after dedisp_stream_sync. */
int dedisp_stream_push(dedisp_stream *s, const void *h_chunk, void **d_out, void **done_event);
/* dedisp_stream_wait_event: make the caller's `stream` (cudaStream_t as void*) wait, on the device,
 * for a done_event returned by dedisp_stream_push, so that work queued on it afterwards may read
 * the block without a host synchronisation. EINVAL on a NULL event. */
int dedisp_stream_wait_event(void *done_event, void *stream);
/* dedisp_stream_release_after: a consumer that reads output blocks on its own stream (after
 * dedisp_stream_wait_event) hands back an event recorded after its last read; every later
 * dedisp_stream_push computes after that event, so a block is never overwritten (nbuffers pushes later)
 * while the consumer is still reading it. Without this call the consumer must finish reading block k
 * before push k + nbuffers is issued (e.g. by dedisp_stream_sync). EINVAL on NULLs. */
int dedisp_stream_release_after(dedisp_stream *s, void *consumer_event);
int dedisp_stream_sync(dedisp_stream *s);
int dedisp_stream_destroy(dedisp_stream *s);

#ifdef __cplusplus
}
#endif
#endif /* DEDISP_B200_H */
