// plan.cu — subsystem (1): the C ABI of include/dedisp.h (plan create / execute / destroy and
// inspection). Host logic only; kernels live in kernels_tiled.cu and subband.cu.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>

#include "plan.h"

namespace {

int fail_cuda(dedisp_plan *p, cudaError_t e, const char *what) {
    if (p) p->cuda_err = std::string(what) + ": " + cudaGetErrorString(e);
    return e == cudaErrorMemoryAllocation ? DEDISP_ENOMEM : DEDISP_ECUDA;
}

int resolve_kernel(const dedisp_plan *p) {
    int k = p->kernel;
    if (k == DEDISP_KERNEL_AUTO) {
        // SUBBAND pays a tile prologue + epilogue per pass worth about 20 channels of its inner loop, TILED
        // runs at a flat ~13 % of the add peak: plans cut into passes shorter than that (the paper-regime
        // sweeps at 250 / 500 channels: 3 and 13 channels per pass) are faster on TILED (profiles/r2_paper_sweep.md)
        const bool short_passes = p->sb.ok && p->tiled.ok &&
                                  (long long)p->nchans * p->sb.nranges < 20ll * (long long)p->sb.passes.size();
        k = p->sb.ok && !short_passes ? DEDISP_KERNEL_SUBBAND : p->tiled.ok ? DEDISP_KERNEL_TILED : DEDISP_KERNEL_NAIVE;
    }
    return k;
}

}  // namespace

int execute_impl(dedisp_plan *p, const void *d_in, long long in_stride, long long nsamp_out, void *d_out,
                 long long out_stride, Batch b, cudaStream_t st, const SbRun &run) {
    if (!p || !d_in || !d_out || nsamp_out < 1) return DEDISP_EINVAL;
    if (in_stride < nsamp_out + p->maxshift || out_stride < nsamp_out) return DEDISP_EINVAL;
    if (p->flags & DEDISP_PLAN_HOST_ONLY) return DEDISP_EUNSUPPORTED;
    if (nsamp_out + p->maxshift >= (1ll << 40)) return DEDISP_EUNSUPPORTED;
    int k = resolve_kernel(p);
    // TILED aligns window starts down to 16 B relative to an aligned base (SUBBAND takes any alignment)
    if (((uintptr_t)d_in & 15) != 0 && k == DEDISP_KERNEL_TILED) {
        if (p->kernel != DEDISP_KERNEL_AUTO) return DEDISP_EINVAL;
        k = DEDISP_KERNEL_NAIVE;
    }
    cudaError_t e;
    switch (k) {
        case DEDISP_KERNEL_SUBBAND: e = launch_subband(p, d_in, in_stride, nsamp_out, d_out, out_stride, b, st, run); break;
        case DEDISP_KERNEL_TILED: e = launch_tiled(p, d_in, in_stride, nsamp_out, d_out, out_stride, b, st); break;
        default: e = launch_naive(p, d_in, in_stride, nsamp_out, d_out, out_stride, b, st); break;
    }
    if (e != cudaSuccess) return fail_cuda(p, e, "kernel launch");
    return DEDISP_OK;
}

extern "C" {

int dedisp_shift_table_host(int nchans, double fch1, double foff, double tsamp, const double *h_dm_list, int ndm,
                            int *h_table, long long *h_maxshift) {
    return build_shift_table(nchans, fch1, foff, tsamp, h_dm_list, ndm, h_table, h_maxshift);
}

int dedisp_plan_create_ex(dedisp_plan **plan, int nchans, double fch1, double foff, double tsamp,
                          const double *h_dm_list, int ndm, int in_dtype, unsigned flags) {
    if (!plan) return DEDISP_EINVAL;
    *plan = nullptr;
    if (in_dtype != DEDISP_U8 && in_dtype != DEDISP_F16 && in_dtype != DEDISP_F32) return DEDISP_EINVAL;
    if (nchans < 1 || ndm < 1 || !h_dm_list) return DEDISP_EINVAL;
    if ((flags & DEDISP_PLAN_TIME_MAJOR) && (in_dtype != DEDISP_U8 || nchans % 16 != 0)) return DEDISP_EINVAL;
    if ((double)nchans * (double)ndm > 2.0e9) return DEDISP_EUNSUPPORTED;
    dedisp_plan *p = new (std::nothrow) dedisp_plan();
    if (!p) return DEDISP_ENOMEM;
    int rc = DEDISP_OK;
    try {
        p->nchans = nchans; p->ndm = ndm; p->dtype = in_dtype;
        p->fch1 = fch1; p->foff = foff; p->tsamp = tsamp; p->flags = flags;
        p->time_major = (flags & DEDISP_PLAN_TIME_MAJOR) != 0;
        p->dm.assign(h_dm_list, h_dm_list + ndm);
        p->shifts.resize((size_t)nchans * ndm);
        rc = build_shift_table(nchans, fch1, foff, tsamp, p->dm.data(), ndm, p->shifts.data(), &p->maxshift);
        if (rc == DEDISP_OK && in_dtype == DEDISP_U8 && (double)nchans * 255.0 > 2147483647.0) rc = DEDISP_EUNSUPPORTED;
        if (rc == DEDISP_OK) {
            tiled_choose_geom(p);
            subband_build(p);
        }
    } catch (const std::bad_alloc &) {
        rc = DEDISP_ENOMEM;
    }
    if (rc != DEDISP_OK) { delete p; return rc; }

    if (!(flags & DEDISP_PLAN_HOST_ONLY)) {
        cudaError_t e = cudaGetDevice(&p->device);
        if (e != cudaSuccess) { rc = fail_cuda(nullptr, e, "cudaGetDevice"); delete p; return rc; }
        cudaDeviceProp prop;
        e = cudaGetDeviceProperties(&prop, p->device);
        if (e != cudaSuccess) { delete p; return DEDISP_ECUDA; }
        if (prop.major != 10) { delete p; return DEDISP_EUNSUPPORTED; }  // sm_100a cubin only, no fallback
        p->sm_count = prop.multiProcessorCount;
        const size_t bytes = p->shifts.size() * sizeof(int32_t);
        e = cudaMalloc(&p->d_shifts, bytes);
        if (e == cudaSuccess) e = cudaMemcpy(p->d_shifts, p->shifts.data(), bytes, cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = subband_upload(p);
        if (e != cudaSuccess) {
            rc = fail_cuda(nullptr, e, "plan upload");
            dedisp_plan_destroy(p);
            return rc;
        }
    }
    *plan = p;
    return DEDISP_OK;
}

int dedisp_plan_create(dedisp_plan **plan, int nchans, double fch1, double foff, double tsamp,
                       const double *h_dm_list, int ndm, int in_dtype) {
    return dedisp_plan_create_ex(plan, nchans, fch1, foff, tsamp, h_dm_list, ndm, in_dtype, DEDISP_PLAN_DEFAULT);
}

int dedisp_execute_strided(dedisp_plan *p, const void *d_in, long long in_stride, long long nsamp_out,
                           void *d_out, long long out_stride, void *stream) {
    return execute_impl(p, d_in, in_stride, nsamp_out, d_out, out_stride, Batch(), (cudaStream_t)stream);
}

int dedisp_execute_time_major(dedisp_plan *p, const void *d_in, int nbits, long long row_bytes, long long nsamp_out,
                              void *d_out, void *stream) {
    if (!p || !d_in || !d_out || nsamp_out < 1) return DEDISP_EINVAL;
    if (nbits != 1 && nbits != 2 && nbits != 4 && nbits != 8) return DEDISP_EINVAL;
    if (row_bytes * 8 < (long long)p->nchans * nbits || (row_bytes & 15) != 0 || ((uintptr_t)d_in & 15) != 0) return DEDISP_EINVAL;
    if (p->flags & DEDISP_PLAN_HOST_ONLY) return DEDISP_EUNSUPPORTED;
    if (!p->time_major || !p->sb.ok || p->sb.cb != 16) return DEDISP_EUNSUPPORTED;   // corner turn lives in the SUBBAND staging step
    if (nsamp_out + p->maxshift >= (1ll << 40)) return DEDISP_EUNSUPPORTED;
    SbRun run;
    run.tm_bits = nbits;
    const cudaError_t e = launch_subband(p, d_in, row_bytes, nsamp_out, d_out, nsamp_out, Batch(), (cudaStream_t)stream, run);
    if (e != cudaSuccess) return fail_cuda(p, e, "kernel launch");
    return DEDISP_OK;
}

int dedisp_execute(dedisp_plan *p, const void *d_in, long long nsamp_out, void *d_out, void *stream) {
    if (!p) return DEDISP_EINVAL;
    return execute_impl(p, d_in, nsamp_out + p->maxshift, nsamp_out, d_out, nsamp_out, Batch(), (cudaStream_t)stream);
}

int dedisp_execute_batched(dedisp_plan *p, int nbeams, const void *d_in, long long in_stride,
                           long long in_beam_stride, long long nsamp_out, void *d_out, long long out_stride,
                           long long out_beam_stride, void *stream) {
    if (!p || nbeams < 1 || nbeams > 65535) return DEDISP_EINVAL;
    if (in_beam_stride < (long long)p->nchans * in_stride - (in_stride - nsamp_out - p->maxshift)) return DEDISP_EINVAL;
    if (out_beam_stride < (long long)p->ndm * out_stride - (out_stride - nsamp_out)) return DEDISP_EINVAL;
    Batch b;
    b.n = nbeams; b.in_stride = in_beam_stride; b.out_stride = out_beam_stride;
    return execute_impl(p, d_in, in_stride, nsamp_out, d_out, out_stride, b, (cudaStream_t)stream);
}

int dedisp_execute_host(dedisp_plan *p, const void *h_in, long long nsamp_out, void *h_out, void *stream) {
    if (!p || !h_in || !h_out || nsamp_out < 1) return DEDISP_EINVAL;
    if (p->flags & DEDISP_PLAN_HOST_ONLY) return DEDISP_EUNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    const long long nsamp_in = nsamp_out + p->maxshift;
    const size_t in_bytes = (size_t)p->nchans * nsamp_in * dtype_esize(p->dtype);
    const size_t out_bytes = (size_t)p->ndm * nsamp_out * 4;
    cudaError_t e = cudaSuccess;
    if (in_bytes > p->host_in_bytes) {
        if (p->d_host_in) cudaFree(p->d_host_in);
        p->d_host_in = nullptr; p->host_in_bytes = 0;
        e = cudaMalloc(&p->d_host_in, in_bytes);
        if (e != cudaSuccess) return fail_cuda(p, e, "dedisp_execute_host input scratch");
        p->host_in_bytes = in_bytes;
    }
    if (out_bytes > p->host_out_bytes) {
        if (p->d_host_out) cudaFree(p->d_host_out);
        p->d_host_out = nullptr; p->host_out_bytes = 0;
        e = cudaMalloc(&p->d_host_out, out_bytes);
        if (e != cudaSuccess) return fail_cuda(p, e, "dedisp_execute_host output scratch");
        p->host_out_bytes = out_bytes;
    }
    // A SUBBAND launch reads only the channels of its own sub-bands (plus at most 15 bytes on either side of a
    // window, which are discarded): copy the channels in the order the launches need them on a second stream
    // and let launch g start as soon as its rows have landed, so that most of the H2D transfer hides under
    // the earlier launches. The launches run last sub-band first (fewest channels: the first launch starts
    // early), so what launch g needs is always a suffix [min c_begin of its passes, nchans) of the channels.
    const int nlaunch = (int)p->sb.launch_begin.size() - 1;
    const bool overlap = resolve_kernel(p) == DEDISP_KERNEL_SUBBAND && nlaunch > 1 && !subband_merges(p);   // a merged launch reads every channel at once
    if (overlap) {
        if (!p->host_copy_st) {
            e = cudaStreamCreateWithFlags(&p->host_copy_st, cudaStreamNonBlocking);
            if (e != cudaSuccess) return fail_cuda(p, e, "dedisp_execute_host copy stream");
        }
        while ((int)p->host_pass_ready.size() < nlaunch) {
            cudaEvent_t ev;
            e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
            if (e != cudaSuccess) return fail_cuda(p, e, "dedisp_execute_host event");
            p->host_pass_ready.push_back(ev);
        }
        cudaEvent_t start = p->host_pass_ready[0];           // order the copy stream after the caller's stream
        e = cudaEventRecord(start, st);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(p->host_copy_st, start, 0);
        const size_t row_bytes = (size_t)nsamp_in * dtype_esize(p->dtype);
        int copied_from = p->nchans;                          // channels [copied_from, nchans) are queued
        for (int i = 0; i < nlaunch && e == cudaSuccess; ++i) {
            const int g = nlaunch - 1 - i;
            int need = p->nchans;
            for (int q = p->sb.launch_begin[g]; q < p->sb.launch_begin[g + 1]; ++q) need = std::min(need, p->sb.passes[q].c_begin);
            if (g == 0) need = 0;
            if (need < copied_from) {
                e = cudaMemcpyAsync((char *)p->d_host_in + need * row_bytes, (const char *)h_in + need * row_bytes,
                                    (size_t)(copied_from - need) * row_bytes, cudaMemcpyHostToDevice, p->host_copy_st);
                copied_from = need;
            }
            if (e == cudaSuccess) e = cudaEventRecord(p->host_pass_ready[g], p->host_copy_st);
        }
        if (e != cudaSuccess) return fail_cuda(p, e, "dedisp_execute_host H2D");
    } else {
        e = cudaMemcpyAsync(p->d_host_in, h_in, in_bytes, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return fail_cuda(p, e, "dedisp_execute_host H2D");
    }
    int rc = DEDISP_OK;
    SbRun run;
    if (overlap) {
        run.pass_ready = p->host_pass_ready.data();
        run.reverse = true;
    }
    p->host_slabs = 0;
    if (overlap && p->sb.nblk >= 4) {
        // ... and run the LAST TWO passes slab by slab over the DM blocks, so that the D2H copy of a finished
        // slab of out rows overlaps the rest of the work. Every output row needs every input channel, so no
        // slab can finish before the H2D copy has: the last pass of the first slab waits for it, and the
        // second-last pass of LOOKAHEAD further slabs is queued in front of it to fill that wait.
        const int NSLAB = std::min(8, p->sb.nblk), LOOKAHEAD = 2;
        if (!p->host_d2h_st) e = cudaStreamCreateWithFlags(&p->host_d2h_st, cudaStreamNonBlocking);
        while (e == cudaSuccess && (int)p->host_slab_done.size() < NSLAB) {
            cudaEvent_t ev;
            e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
            if (e == cudaSuccess) p->host_slab_done.push_back(ev);
        }
        if (e != cudaSuccess) return fail_cuda(p, e, "dedisp_execute_host slabs");
        const int npass = nlaunch;                           // launches, in the order they run
        const int nslabbed = npass >= 3 ? 2 : 1;             // launches (the last ones to run) done slab by slab
        run.pass_lo = 0; run.pass_hi = npass - nslabbed;     // the others over the whole grid
        rc = execute_impl(p, p->d_host_in, nsamp_in, nsamp_out, p->d_host_out, nsamp_out, Batch(), st, run);
        auto slab_pass = [&](int i, int sl) -> int {         // launch-order pass i on DM slab sl
            SbRun r = run;
            r.pass_lo = i; r.pass_hi = i + 1;
            r.blk_lo = (int)((long long)p->sb.nblk * sl / NSLAB);
            r.blk_hi = (int)((long long)p->sb.nblk * (sl + 1) / NSLAB);
            return execute_impl(p, p->d_host_in, nsamp_in, nsamp_out, p->d_host_out, nsamp_out, Batch(), st, r);
        };
        if (nslabbed == 2)
            for (int sl = 0; sl < std::min(LOOKAHEAD, NSLAB) && rc == DEDISP_OK; ++sl) rc = slab_pass(npass - 2, sl);
        for (int sl = 0; sl < NSLAB && rc == DEDISP_OK; ++sl) {
            rc = slab_pass(npass - 1, sl);
            if (rc != DEDISP_OK) break;
            ++p->host_slabs;
            const long long d0 = std::min<long long>(p->ndm, (long long)((long long)p->sb.nblk * sl / NSLAB) * SB_ROWS);
            const long long d1 = std::min<long long>(p->ndm, (long long)((long long)p->sb.nblk * (sl + 1) / NSLAB) * SB_ROWS);
            e = cudaEventRecord(p->host_slab_done[sl], st);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(p->host_d2h_st, p->host_slab_done[sl], 0);
            if (e == cudaSuccess && d1 > d0)
                e = cudaMemcpyAsync((char *)h_out + d0 * nsamp_out * 4, (char *)p->d_host_out + d0 * nsamp_out * 4,
                                    (size_t)(d1 - d0) * nsamp_out * 4, cudaMemcpyDeviceToHost, p->host_d2h_st);
            if (e != cudaSuccess) { rc = fail_cuda(p, e, "dedisp_execute_host slab D2H"); break; }
            if (nslabbed == 2 && sl + LOOKAHEAD < NSLAB) rc = slab_pass(npass - 2, sl + LOOKAHEAD);
        }
        if (rc != DEDISP_OK) return rc;
        e = cudaStreamSynchronize(p->host_d2h_st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return fail_cuda(p, e, "dedisp_execute_host D2H");
        return DEDISP_OK;
    }
    rc = execute_impl(p, p->d_host_in, nsamp_in, nsamp_out, p->d_host_out, nsamp_out, Batch(), st, run);
    if (rc != DEDISP_OK) return rc;
    e = cudaMemcpyAsync(h_out, p->d_host_out, out_bytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail_cuda(p, e, "dedisp_execute_host D2H");
    return DEDISP_OK;
}

int dedisp_plan_destroy(dedisp_plan *p) {
    if (!p) return DEDISP_OK;
    if (p->d_shifts) cudaFree(p->d_shifts);
    if (p->d_host_in) cudaFree(p->d_host_in);
    if (p->d_host_out) cudaFree(p->d_host_out);
    for (cudaEvent_t ev : p->host_pass_ready) cudaEventDestroy(ev);
    if (p->host_copy_st) cudaStreamDestroy(p->host_copy_st);
    for (cudaEvent_t ev : p->host_slab_done) cudaEventDestroy(ev);
    if (p->host_d2h_st) cudaStreamDestroy(p->host_d2h_st);
    subband_free(p);
    delete p;
    return DEDISP_OK;
}

long long dedisp_plan_max_shift(const dedisp_plan *p) { return p ? p->maxshift : -1; }
int dedisp_plan_nchans(const dedisp_plan *p) { return p ? p->nchans : -1; }
int dedisp_plan_ndm(const dedisp_plan *p) { return p ? p->ndm : -1; }

int dedisp_plan_get_shifts(const dedisp_plan *p, int *h_out) {
    if (!p || !h_out) return DEDISP_EINVAL;
    std::memcpy(h_out, p->shifts.data(), p->shifts.size() * sizeof(int32_t));
    return DEDISP_OK;
}

int dedisp_plan_set_kernel(dedisp_plan *p, int kernel) {
    if (!p) return DEDISP_EINVAL;
    switch (kernel) {
        case DEDISP_KERNEL_AUTO:
        case DEDISP_KERNEL_NAIVE: break;
        case DEDISP_KERNEL_TILED: if (!p->tiled.ok) return DEDISP_EUNSUPPORTED; break;
        case DEDISP_KERNEL_SUBBAND: if (!p->sb.ok) return DEDISP_EUNSUPPORTED; break;
        default: return DEDISP_EINVAL;
    }
    p->kernel = kernel;
    return DEDISP_OK;
}

int dedisp_plan_set_pass_merge(dedisp_plan *p, int on) {
    if (!p) return DEDISP_EINVAL;
    p->merge_fp_passes = on != 0;
    return DEDISP_OK;
}

int dedisp_plan_get_kernel(const dedisp_plan *p) { return p ? resolve_kernel(p) : -1; }

int dedisp_plan_num_subbands(const dedisp_plan *p) {
    if (!p) return -1;
    if (!p->sb.ok) return 0;
    int n = 0;   // sub-bands of the first DM range (plans with a changing DM step have one partition per range)
    for (const SubbandPass &ps : p->sb.passes) n += ps.blk_begin == 0;
    return n;
}

int dedisp_plan_get_subbands(const dedisp_plan *p, int *h_first_chan) {
    if (!p || !h_first_chan) return DEDISP_EINVAL;
    if (!p->sb.ok) return DEDISP_EUNSUPPORTED;
    int n = 0;
    for (const SubbandPass &ps : p->sb.passes)
        if (ps.blk_begin == 0) h_first_chan[n++] = ps.c_begin;
    h_first_chan[n] = p->nchans;
    return DEDISP_OK;
}

long long dedisp_plan_verify_records(const dedisp_plan *p) {
    if (!p || !p->sb.ok) return -1;
    return subband_verify_records(p);
}

int dedisp_plan_get_geometry(const dedisp_plan *p, int *h_out) {
    if (!p || !h_out) return DEDISP_EINVAL;
    const SubbandGeom &sb = p->sb;
    const int v[8] = {sb.ok ? sb.cb : 0, sb.ok ? sb.cb_raw : 0, sb.slot_chunks * 16, (int)sb.smem, (int)sb.smem_raw,
                      sb.nblk, sb.nranges, (int)sb.passes.size()};
    std::memcpy(h_out, v, sizeof v);
    return DEDISP_OK;
}

int dedisp_plan_last_host_slabs(const dedisp_plan *p) { return p ? p->host_slabs : -1; }

int dedisp_plan_launches_per_execute(const dedisp_plan *p) {
    if (!p) return -1;
    return subband_launches(p, resolve_kernel(p));
}

const char *dedisp_error_string(int code) {
    switch (code) {
        case DEDISP_OK: return "ok";
        case DEDISP_EINVAL: return "invalid argument";
        case DEDISP_ENOMEM: return "out of memory";
        case DEDISP_ECUDA: return "CUDA error";
        case DEDISP_EUNSUPPORTED: return "unsupported (device is not sm_100, shift >= 2^31, host-only plan, or kernel not admitted by the plan)";
        case DEDISP_ETOOLARGE: return "size exceeds the fixed scratch of a no-allocation entry point (dedisp_detect_static: ndm > DEDISP_DETECT_STATIC_MAX_NDM)";
        default: return "unknown error code";
    }
}

const char *dedisp_last_cuda_error(const dedisp_plan *p) { return p ? p->cuda_err.c_str() : ""; }

}  // extern "C"
