// subband.cu — SUBBAND kernel (exact sub-band re-skewed multi-pass with register-window reuse).
//
// Not built yet: subband_build() leaves p->sb.ok = false, so AUTO resolves to the TILED kernel and
// dedisp_plan_set_kernel(DEDISP_KERNEL_SUBBAND) returns DEDISP_EUNSUPPORTED. The entry points exist
// so that the plan code and the ABI are stable.
#include "plan.h"

void subband_build(dedisp_plan *p) { p->sb = SubbandGeom(); }

cudaError_t subband_upload(dedisp_plan *) { return cudaSuccess; }

void subband_free(dedisp_plan *p) {
    if (p->sb.d_records) cudaFree(p->sb.d_records);
    if (p->sb.d_cta_meta) cudaFree(p->sb.d_cta_meta);
    if (p->sb.d_skew) cudaFree(p->sb.d_skew);
    p->sb.d_records = nullptr;
    p->sb.d_cta_meta = nullptr;
    p->sb.d_skew = nullptr;
}

long long subband_verify_records(const dedisp_plan *) { return -1; }

cudaError_t launch_subband(const dedisp_plan *, const void *, long long, long long, void *, long long, Batch,
                           cudaStream_t) {
    return cudaErrorNotSupported;
}
