// stream.cu — subsystem (4): streaming multi-beam driver (the role the
// MDSM wrapper plays in the paper, §1; BASELINE.json:north_star (4), configs[4]).
//
// Device layout per buffer b (nbuffers >= 2, round-robin over pushes):
//   in [b] : [beam][chan][row]  with row = maxshift + chunk samples (padded to a 16-byte multiple);
//            columns [0, maxshift) hold the history carried from the previous chunk, columns
//            [maxshift, maxshift + chunk) the chunk just copied from the host.
//   out[b] : [beam][dm][chunk]  int32 (u8 input) or float32.
// Push k on the COPY stream: wait until the compute that last read in[b] is done; fill the history
// (zeros for k = 0, else a strided device copy of the last maxshift columns of buffer k-1); one
// cudaMemcpy2DAsync host -> device for all beams and channels; record h2d_done[b].
// On the COMPUTE stream: wait h2d_done[b]; one batched launch over all beams; record done[b].
// Copy k+1 therefore overlaps compute k; nothing is exchanged between chunks but the read-only
// history columns.
#include <new>

#include "plan.h"

struct dedisp_stream {
    dedisp_plan *plan = nullptr;
    int nbeams = 0, nbuf = 0, esize = 0;
    long long chunk = 0, row = 0;  // row: device input row stride in elements
    long long pushes = 0;
    cudaStream_t copy_st = nullptr, comp_st = nullptr;
    std::vector<void *> d_in, d_out;
    std::vector<cudaEvent_t> h2d_done, done;
};

namespace {

int stream_fail(dedisp_stream *s, cudaError_t e, const char *what) {
    s->plan->cuda_err = std::string(what) + ": " + cudaGetErrorString(e);
    return e == cudaErrorMemoryAllocation ? DEDISP_ENOMEM : DEDISP_ECUDA;
}

}  // namespace

extern "C" {

int dedisp_stream_destroy(dedisp_stream *s) {
    if (!s) return DEDISP_OK;
    if (s->copy_st) cudaStreamSynchronize(s->copy_st);
    if (s->comp_st) cudaStreamSynchronize(s->comp_st);
    for (void *p : s->d_in) if (p) cudaFree(p);
    for (void *p : s->d_out) if (p) cudaFree(p);
    for (cudaEvent_t e : s->h2d_done) if (e) cudaEventDestroy(e);
    for (cudaEvent_t e : s->done) if (e) cudaEventDestroy(e);
    if (s->copy_st) cudaStreamDestroy(s->copy_st);
    if (s->comp_st) cudaStreamDestroy(s->comp_st);
    delete s;
    return DEDISP_OK;
}

int dedisp_stream_create(dedisp_stream **out, dedisp_plan *plan, int nbeams, long long chunk_nsamp, int nbuffers) {
    if (!out) return DEDISP_EINVAL;
    *out = nullptr;
    if (!plan || nbeams < 1 || nbeams > 65535 || chunk_nsamp < 1 || nbuffers < 2 || nbuffers > 16) return DEDISP_EINVAL;
    if (plan->flags & DEDISP_PLAN_HOST_ONLY) return DEDISP_EUNSUPPORTED;
    dedisp_stream *s = new (std::nothrow) dedisp_stream();
    if (!s) return DEDISP_ENOMEM;
    s->plan = plan;
    s->nbeams = nbeams;
    s->nbuf = nbuffers;
    s->esize = dtype_esize(plan->dtype);
    s->chunk = chunk_nsamp;
    const long long per16 = 16 / s->esize;
    s->row = ((plan->maxshift + chunk_nsamp + per16 - 1) / per16) * per16;
    s->d_in.assign(nbuffers, nullptr);
    s->d_out.assign(nbuffers, nullptr);
    s->h2d_done.assign(nbuffers, nullptr);
    s->done.assign(nbuffers, nullptr);
    const size_t in_bytes = (size_t)nbeams * plan->nchans * s->row * s->esize;
    const size_t out_bytes = (size_t)nbeams * plan->ndm * chunk_nsamp * 4;
    cudaError_t e = cudaStreamCreateWithFlags(&s->copy_st, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&s->comp_st, cudaStreamNonBlocking);
    for (int b = 0; b < nbuffers && e == cudaSuccess; ++b) {
        e = cudaMalloc(&s->d_in[b], in_bytes);
        if (e == cudaSuccess) e = cudaMalloc(&s->d_out[b], out_bytes);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->h2d_done[b], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->done[b], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) {
        const int rc = stream_fail(s, e, "dedisp_stream_create");
        dedisp_stream_destroy(s);
        return rc;
    }
    *out = s;
    return DEDISP_OK;
}

int dedisp_stream_push(dedisp_stream *s, const void *h_chunk, void **d_out, void **done_event) {
    if (!s || !h_chunk) return DEDISP_EINVAL;
    dedisp_plan *p = s->plan;
    const int b = (int)(s->pushes % s->nbuf);
    const long long rows = (long long)s->nbeams * p->nchans;
    const size_t pitch = (size_t)s->row * s->esize;
    const size_t hist = (size_t)p->maxshift * s->esize;
    char *dst = (char *)s->d_in[b];
    cudaError_t e = cudaSuccess;
    if (s->pushes >= s->nbuf) e = cudaStreamWaitEvent(s->copy_st, s->done[b], 0);
    if (e == cudaSuccess && hist) {
        if (s->pushes == 0) {
            e = cudaMemset2DAsync(dst, pitch, 0, hist, (size_t)rows, s->copy_st);
        } else {
            const char *prev = (const char *)s->d_in[(s->pushes - 1) % s->nbuf];
            e = cudaMemcpy2DAsync(dst, pitch, prev + (size_t)s->chunk * s->esize, pitch, hist, (size_t)rows,
                                  cudaMemcpyDeviceToDevice, s->copy_st);
        }
    }
    if (e == cudaSuccess)
        e = cudaMemcpy2DAsync(dst + hist, pitch, h_chunk, (size_t)s->chunk * s->esize, (size_t)s->chunk * s->esize,
                              (size_t)rows, cudaMemcpyHostToDevice, s->copy_st);
    if (e == cudaSuccess) e = cudaEventRecord(s->h2d_done[b], s->copy_st);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(s->comp_st, s->h2d_done[b], 0);
    if (e != cudaSuccess) return stream_fail(s, e, "dedisp_stream_push copy");
    Batch bt;
    bt.n = s->nbeams;
    bt.in_stride = (long long)p->nchans * s->row;
    bt.out_stride = (long long)p->ndm * s->chunk;
    const int rc = execute_impl(p, s->d_in[b], s->row, s->chunk, s->d_out[b], s->chunk, bt, s->comp_st);
    if (rc != DEDISP_OK) return rc;
    e = cudaEventRecord(s->done[b], s->comp_st);
    if (e != cudaSuccess) return stream_fail(s, e, "dedisp_stream_push record");
    if (d_out) *d_out = s->d_out[b];
    if (done_event) *done_event = (void *)s->done[b];
    ++s->pushes;
    return DEDISP_OK;
}

int dedisp_stream_wait_event(void *done_event, void *stream) {
    if (!done_event) return DEDISP_EINVAL;
    return cudaStreamWaitEvent((cudaStream_t)stream, (cudaEvent_t)done_event, 0) == cudaSuccess ? DEDISP_OK : DEDISP_ECUDA;
}

int dedisp_stream_release_after(dedisp_stream *s, void *consumer_event) {
    if (!s || !consumer_event) return DEDISP_EINVAL;
    // every later launch on the compute stream (i.e. every later overwrite of an output block) is
    // ordered after the consumer's event
    const cudaError_t e = cudaStreamWaitEvent(s->comp_st, (cudaEvent_t)consumer_event, 0);
    return e == cudaSuccess ? DEDISP_OK : stream_fail(s, e, "dedisp_stream_release_after");
}

int dedisp_stream_sync(dedisp_stream *s) {
    if (!s) return DEDISP_EINVAL;
    cudaError_t e = cudaStreamSynchronize(s->copy_st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->comp_st);
    if (e != cudaSuccess) return stream_fail(s, e, "dedisp_stream_sync");
    return DEDISP_OK;
}

}  // extern "C"
