// shift_table.cpp — subsystem (2): the per-(channel, DM) integer delays, built once per plan on
// the host in IEEE double ("the shifting value is calculated
// using as few operations as possible" — here it is not calculated in the kernel at all).
//
// Formula (BASELINE.json:north_star; readings R1-R6):
//     s(c,d) = floor( 4.148808e3 * DM_d * (f_c^-2 - f_top^-2) / tsamp + 0.5 ),
//     f_c = fch1 + c*foff (MHz), f_top = fch1, tsamp in s.
// float32 evaluation mis-rounds thousands of entries on the survey configs,
// so this file must be compiled as host code with -ffp-contract=off.
//
// This file shares nothing with oracle/: the expression below is this library's own statement of
// the north_star formula (the per-channel factor is hoisted; the tests check that it agrees with
// the oracle's table on every entry of all five configs).
#include <cmath>
#include <cstdint>

#include "plan.h"

static const double kDispersionConstant = 4.148808e3;  // MHz^2 pc^-1 cm^3 s

int build_shift_table(int nchans, double fch1, double foff, double tsamp, const double *dm, int ndm,
                      int32_t *table, long long *maxshift) {
    if (nchans < 1 || ndm < 1 || !dm || !table) return DEDISP_EINVAL;
    if (!(tsamp > 0.0) || !(fch1 > 0.0) || !(foff < 0.0) || !std::isfinite(tsamp) || !std::isfinite(fch1) ||
        !std::isfinite(foff))
        return DEDISP_EINVAL;
    const double f_low = fch1 + (double)(nchans - 1) * foff;
    if (!(f_low > 0.0)) return DEDISP_EINVAL;
    for (int d = 0; d < ndm; ++d) {
        if (!std::isfinite(dm[d]) || dm[d] < 0.0) return DEDISP_EINVAL;
        if (d > 0 && dm[d] < dm[d - 1]) return DEDISP_EINVAL;  // kernels rely on s non-decreasing in d
    }
    const double inv_top2 = 1.0 / (fch1 * fch1);
    long long mx = 0;
    for (int c = 0; c < nchans; ++c) {
        const double f = fch1 + (double)c * foff;
        const double dinv = 1.0 / (f * f) - inv_top2;  // f_c^-2 - f_top^-2
        int32_t *row = table + (size_t)c * ndm;
        for (int d = 0; d < ndm; ++d) {
            const double x = ((kDispersionConstant * dm[d]) * dinv) / tsamp;
            const double r = std::floor(x + 0.5);
            if (!(r < 2147483648.0)) return DEDISP_EUNSUPPORTED;
            const long long s = (long long)r;
            row[d] = (int32_t)s;
            if (s > mx) mx = s;
        }
    }
    if (maxshift) *maxshift = mx;
    return DEDISP_OK;
}
