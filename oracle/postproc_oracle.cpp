// ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path.
//
// Plain, slow CPU implementation of the thesis' post-processing of the dedispersed time series
// and of the first stage of event detection (§3.5 "Signal Post-processing"
// and §3.6 "Detection and Candidate Selection"), one function per step, each in the paper's
// order and notation, double precision throughout.  Shares no code with the CUDA library.
//
//   1. median filtering (eq 3.4):  y_m = median{ x_i, i in w },  w a
//      neighbourhood of odd length centred on m ("A w value of 5 or 7 generally gives a good
//      ratio");
//   2. detrending: subtract the best-fit line found by linear regression over the
//      whole series (first pass: regression parameters; second pass: subtract, and accumulate
//      the standard deviation);
//   3. normalisation ("by adding a third pass the data can be normalised"): divide
//      by that standard deviation;
//   4. thresholding: keep the samples above n sigma as (time, DM, intensity)
//      triplets, one list per beam.
//
// Readings where the paper is silent (R15-R19):
//   R15 window at the ends of the series: indices are clamped to [0, n-1] (edge replication), so
//       every output is the median of exactly w values and is one of the inputs;
//   R16 regression abscissa: the sample index t = 0 .. n-1; ordinary least squares;
//   R17 standard deviation: population form, sigma^2 = (1/n) sum r_t^2 of the detrended series r
//       (its mean is zero by construction); sigma = 0 (constant series) gives all-zero output;
//   R18 threshold: strict, value > n sigma, the value being the normalised sample (units of sigma);
//       without normalisation the comparison is r_t > n * sigma with the same sigma;
//   R19 order: median filter, then detrend, then normalise, then threshold (the order of §3.5-3.6).
//
// Pins (tests/test_postproc_pins.py, all `-m "not gpu"`): numpy's median over edge-padded sliding
// windows; hand-worked windows; idempotence on monotone ramps; spike removal; numpy.polyfit for
// the regression line; an exact line detrends to zeros; closed-form sigma of known sequences;
// output mean 0 / variance 1; the Fig 2.6 recipe (amplitude 0.25 over 1024
// channels = S/N 8) crossing a 6 sigma threshold at the injected (DM, t) only.
// No function here is "parity unpinned".

#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <vector>

extern "C" {

// eq 3.4 with the median as the operation; window of odd length w centred on m, ends clamped (R15).
void oracle_median_filter(const double* x, int64_t n, int w, double* y)
{
    const int h = (w - 1) / 2;
    std::vector<double> win((size_t)w);
    for (int64_t m = 0; m < n; ++m) {
        for (int i = -h; i <= h; ++i) {
            int64_t j = m + i;
            if (j < 0) j = 0;
            if (j > n - 1) j = n - 1;
            win[(size_t)(i + h)] = x[j];
        }
        std::sort(win.begin(), win.end());
        y[m] = win[(size_t)h];
    }
}

// First pass of the detrending: ordinary least squares of y_t on t = 0..n-1.
// Textbook normal equations:  slope = (n Sxy - Sx Sy) / (n Sxx - Sx^2),  intercept = (Sy - slope Sx) / n.
void oracle_fit_line(const double* y, int64_t n, double* intercept, double* slope)
{
    double sx = 0.0, sy = 0.0, sxx = 0.0, sxy = 0.0;
    for (int64_t t = 0; t < n; ++t) {
        const double x = (double)t;
        sx += x;
        sy += y[t];
        sxx += x * x;
        sxy += x * y[t];
    }
    const double den = (double)n * sxx - sx * sx;
    *slope = den != 0.0 ? ((double)n * sxy - sx * sy) / den : 0.0;     // n = 1: no slope
    *intercept = (sy - *slope * sx) / (double)n;
}

// Second pass: subtract the trend line, and accumulate the standard deviation (R17).
void oracle_detrend(const double* y, int64_t n, double intercept, double slope, double* r, double* sigma)
{
    double ss = 0.0;
    for (int64_t t = 0; t < n; ++t) {
        r[t] = y[t] - (intercept + slope * (double)t);
        ss += r[t] * r[t];
    }
    *sigma = std::sqrt(ss / (double)n);
}

// Third pass: normalise (sigma = 0 gives zeros, R17).
void oracle_normalise(const double* r, int64_t n, double sigma, double* z)
{
    for (int64_t t = 0; t < n; ++t) z[t] = sigma > 0.0 ? r[t] / sigma : 0.0;
}

// The whole of §3.5 on a set of series (rows), OpenMP over the rows only.  x: float32 or int32
// series [nrows][stride] (is_int selects), the output of the dedispersion stage.  median_window
// <= 1 skips step 1; detrend = 0 stops after step 1 (normalise must then be 0 too: the paper
// normalises only the detrended series); normalise = 0 stops after step 2.  z: double [nrows][n]
// processed series; stats: double [nrows][3] = (intercept, slope, sigma) of steps 2-3 (zeros
// without detrending), may be null.
void oracle_postprocess_rows(const void* x, int is_int, int64_t nrows, int64_t n, int64_t stride,
                             int median_window, int detrend, int normalise, double* z, double* stats)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t row = 0; row < nrows; ++row) {
        std::vector<double> a((size_t)n), b((size_t)n);
        for (int64_t t = 0; t < n; ++t)
            a[(size_t)t] = is_int ? (double)((const int32_t*)x)[row * stride + t]
                                  : (double)((const float*)x)[row * stride + t];
        if (median_window > 1) {
            oracle_median_filter(a.data(), n, median_window, b.data());
            a.swap(b);
        }
        double intercept = 0.0, slope = 0.0, sigma = 0.0;
        double* out = z + row * n;
        if (detrend) {
            oracle_fit_line(a.data(), n, &intercept, &slope);
            oracle_detrend(a.data(), n, intercept, slope, b.data(), &sigma);
            if (normalise) oracle_normalise(b.data(), n, sigma, out);
            else
                for (int64_t t = 0; t < n; ++t) out[t] = b[(size_t)t];
        } else {
            for (int64_t t = 0; t < n; ++t) out[t] = a[(size_t)t];
        }
        if (stats) {
            stats[row * 3 + 0] = intercept;
            stats[row * 3 + 1] = slope;
            stats[row * 3 + 2] = sigma;
        }
    }
}

// §3.6 first stage: (time, DM, intensity) triplets of the samples above n sigma (R18), per beam.
// z: [nbeams][ndm][n] processed series; sigma_or_null: per-row sigma when z is NOT normalised
// (then the test is z > nsigma * sigma), null when it is.  Writes up to `capacity` entries in
// (beam, dm, t) order and returns the total number found.
int64_t oracle_threshold(const double* z, int nbeams, int ndm, int64_t n, double nsigma,
                         const double* sigma_or_null, int32_t* beam_out, int32_t* dm_out, int64_t* t_out,
                         double* value_out, int64_t capacity)
{
    int64_t count = 0;
    for (int b = 0; b < nbeams; ++b)
        for (int d = 0; d < ndm; ++d) {
            const int64_t row = (int64_t)b * ndm + d;
            const double level = sigma_or_null ? nsigma * sigma_or_null[row] : nsigma;
            for (int64_t t = 0; t < n; ++t) {
                const double v = z[row * n + t];
                if (v > level) {
                    if (count < capacity) {
                        beam_out[count] = b;
                        dm_out[count] = d;
                        t_out[count] = t;
                        value_out[count] = v;
                    }
                    ++count;
                }
            }
        }
    return count;
}

}  // extern "C"
