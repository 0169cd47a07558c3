// Host shift-table builder.  Plain C++, double precision, compiled with
// -ffp-contract=off.  Written from PAPER.md eq 2.2/2.3 with the constant of
// eq 1.14; it shares no code with oracle/ -- a test asserts the two tables agree.
//
//   DeltaT(c) uses (nu0 + c*dnu)^-2 - nu0^-2 with nu0 = fch1 = channel 0,
//   Delta t(d,c) = round(DM(d) * DeltaT(c))
//
// The expression is evaluated in the association DESIGN.md reading R5 fixes:
//   x = 4148.808 * DM * (1/(fc*fc) - 1/(fch1*fch1)) / tsamp ;  s = floor(x + 0.5)
// Trials are processed in ascending DM order (the thesis assumes ascending DMs inside a block,
// PAPER.md:972); `order` maps the sorted position back to the caller's row.
#include <algorithm>
#include <cmath>
#include <numeric>

#include "dd_internal.h"

namespace dd {

static const double kDispersionConstant = 4148.808;   // MHz^2 pc^-1 cm^3 s, eq 1.14

static int check_args(int nchans, double fch1, double foff, double tsamp, const double* dm_list,
                      int ndm)
{
    if (nchans < 1) return fail(DD_ERR_BAD_ARG, "nchans must be >= 1");
    if (ndm < 0) return fail(DD_ERR_BAD_ARG, "ndm must be >= 0");
    if (ndm > 0 && !dm_list) return fail(DD_ERR_BAD_ARG, "dm_list is null");
    if (!(tsamp > 0.0) || !std::isfinite(tsamp)) return fail(DD_ERR_BAD_ARG, "tsamp must be > 0");
    if (!(fch1 > 0.0) || !std::isfinite(fch1)) return fail(DD_ERR_BAD_ARG, "fch1 must be > 0");
    if (!std::isfinite(foff) || foff > 0.0)
        return fail(DD_ERR_BAD_ARG, "foff must be <= 0 (channel 0 is the top of the band)");
    double fbottom = fch1 + (double)(nchans - 1) * foff;
    if (!(fbottom > 0.0)) return fail(DD_ERR_BAD_ARG, "lowest channel frequency must be > 0");
    for (int d = 0; d < ndm; ++d)
        if (!std::isfinite(dm_list[d]) || dm_list[d] < 0.0)
            return fail(DD_ERR_BAD_ARG, "DM values must be finite and >= 0");
    return DD_OK;
}

// delay of channel `chan` at dispersion measure `dm`, whole samples, as a double
static inline double delay_samples(double dm, int chan, double fch1, double foff, double tsamp)
{
    const double fc = fch1 + (double)chan * foff;
    const double inv2_c = 1.0 / (fc * fc);
    const double inv2_ref = 1.0 / (fch1 * fch1);
    const double x = kDispersionConstant * dm * (inv2_c - inv2_ref) / tsamp;
    return std::floor(x + 0.5);
}

static const double kShiftLimit = 1073741823.0;   // INT32_MAX / 2

int64_t host_max_shift(int nchans, double fch1, double foff, double tsamp, const double* dm_list,
                       int ndm)
{
    int rc = check_args(nchans, fch1, foff, tsamp, dm_list, ndm);
    if (rc != DD_OK) return rc;
    // s is monotone in DM and in c (1/f^2 grows down the band), so the corner is the maximum;
    // scan the last channel over all trials anyway (cheap) rather than rely on the DM order.
    double best = 0.0;
    for (int d = 0; d < ndm; ++d)
        best = std::max(best, delay_samples(dm_list[d], nchans - 1, fch1, foff, tsamp));
    if (best > kShiftLimit) return fail(DD_ERR_BAD_ARG, "shift exceeds INT32_MAX/2 samples");
    return (int64_t)best;
}

int build_host_table(int nchans, double fch1, double foff, double tsamp, const double* dm_list,
                     int ndm, HostTable* out)
{
    int rc = check_args(nchans, fch1, foff, tsamp, dm_list, ndm);
    if (rc != DD_OK) return rc;
    out->nchans = nchans;
    out->ndm = ndm;
    out->order.resize(ndm);
    std::iota(out->order.begin(), out->order.end(), 0);
    std::stable_sort(out->order.begin(), out->order.end(),
                     [&](int32_t a, int32_t b) { return dm_list[a] < dm_list[b]; });
    out->shift.assign((size_t)ndm * nchans, 0);
    out->maxshift = 0;
    for (int r = 0; r < ndm; ++r) {
        const double dm = dm_list[out->order[r]];
        int32_t* row = &out->shift[(size_t)r * nchans];
        for (int c = 0; c < nchans; ++c) {
            double s = delay_samples(dm, c, fch1, foff, tsamp);
            if (s > kShiftLimit) return fail(DD_ERR_BAD_ARG, "shift exceeds INT32_MAX/2 samples");
            if (s < 0.0) s = 0.0;   // cannot happen for foff <= 0; guards -0.0 / rounding only
            row[c] = (int32_t)s;
            if (row[c] > out->maxshift) out->maxshift = row[c];
        }
    }
    return DD_OK;
}

int64_t max_tile_spread(const HostTable& t, int kb)
{
    int64_t worst = 0;
    for (int r0 = 0; r0 < t.ndm; r0 += kb) {
        int r1 = std::min(t.ndm, r0 + kb) - 1;
        const int32_t* a = &t.shift[(size_t)r0 * t.nchans];
        const int32_t* b = &t.shift[(size_t)r1 * t.nchans];
        for (int c = 0; c < t.nchans; ++c) worst = std::max<int64_t>(worst, (int64_t)b[c] - a[c]);
    }
    return worst;
}

}  // namespace dd
