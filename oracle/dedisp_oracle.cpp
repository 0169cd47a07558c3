// ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path.
//
// Plain, slow, obviously-correct CPU implementation of direct (brute-force)
// incoherent dedispersion, written from the thesis text, sharing no
// code, header, table or helper with the CUDA library under
// paper_1401_8258_b200/.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load this file's shared object.
//
// What it computes (§2.1.1, eq 2.1-2.3; constant eq 1.14,
// PAPER.md:425; delay relation eq 1.15):
//
//     D[d][t] = sum_{c=0}^{nchans-1} X[c][ t + s(d,c) ]                (eq 2.1)
//     s(d,c)  = round( DM_d * DeltaT(c) ),
//     DeltaT(c) = k_DM/t_samp * ( (nu0 + c*dnu)^-2 - nu0^-2 )          (eq 2.2/2.3)
//
// with k_DM = 4148.808 (MHz^2 pc^-1 cm^3 s, eq 1.14), frequencies in MHz,
// t_samp in seconds, nu0 = fch1 = channel 0 = the reference frequency ("usually
// the top frequency"), dnu = foff <= 0, and round(x) taken as
// floor(x + 0.5) (reading R2).  The expression is evaluated in
// double precision exactly in the association written in oracle_shift() below
// (reading R5); compile with -ffp-contract=off.
//
// Layout ("stored in channel order, with time changing the
// fastest"; PAPER.md:1202 buffer holds nsamp + maxshift spectra):
//     X : [nchans][in_stride], in_stride >= nsamp + maxshift, time fastest
//     D : [ndm][nsamp], time fastest
// nsamp is the number of OUTPUT samples per DM trial (reading R7).
//
// Loop nest: literal (d, t, c) with a double accumulator, channels added in
// the order c = 0, 1, 2, ...  Each trial d first fills its own row s[c] of the
// delay table (the thesis computes the table once up front);
// OpenMP parallelises the outermost d loop only.
//
// Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): literal brute force
// written separately in Python on tiny inputs; the paper's printed delay
// constant (eq 1.12/1.14) and the DM_max = 826.5 ~ "827" cross-check of
// eq 6.2 / Table 6.7; DM = 0 row = channel sum;
// nchans = 1 identity; impulse response; monotonicity of s; golden shift
// values under tests/golden/ ; the Fig 2.6 S/N recipe; the
// interchanged (d, c, t) variants at the end of this file are pinned bit for bit
// to the literal nest.  No function here is "parity unpinned".

#include <cmath>
#include <cstdint>
#include <cstddef>
#include <vector>

extern "C" {

// eq 2.2/2.3 with the constant of eq 1.14.
// Returns the delay of channel c at dispersion measure dm, in whole samples.
int64_t oracle_shift(double dm, int c, double fch1, double foff, double tsamp)
{
    double fc = fch1 + (double)c * foff;
    double x = 4148.808 * dm * (1.0 / (fc * fc) - 1.0 / (fch1 * fch1)) / tsamp;
    return (int64_t)std::floor(x + 0.5);
}

// Full table, [ndm][nchans], DM-major.
void oracle_shift_table(int nchans, double fch1, double foff, double tsamp,
                        const double* dm_list, int ndm, int64_t* table)
{
    for (int d = 0; d < ndm; ++d)
        for (int c = 0; c < nchans; ++c)
            table[(size_t)d * nchans + c] = oracle_shift(dm_list[d], c, fch1, foff, tsamp);
}

// maxshift = largest delay over all trials and channels.
int64_t oracle_max_shift(int nchans, double fch1, double foff, double tsamp,
                         const double* dm_list, int ndm)
{
    int64_t m = 0;
    for (int d = 0; d < ndm; ++d)
        for (int c = 0; c < nchans; ++c) {
            int64_t s = oracle_shift(dm_list[d], c, fch1, foff, tsamp);
            if (s > m) m = s;
        }
    return m;
}

// float32 input.  D (double) gets the sums; A (double, may be null) gets
// sum_c |X[c][t+s]|, the scale of the float tolerance in north_star.
// Only the DM rows listed in `rows` (nrows indices into dm_list) are computed;
// output row r of D/A corresponds to dm_list[rows[r]].  rows == null => all.
void oracle_dedisperse_f32(const float* X, int nchans, int64_t nsamp, int64_t in_stride,
                           double fch1, double foff, double tsamp,
                           const double* dm_list, int ndm,
                           const int* rows, int nrows,
                           double* D, double* A)
{
    int nr = rows ? nrows : ndm;
#pragma omp parallel for schedule(dynamic, 1)
    for (int r = 0; r < nr; ++r) {
        int d = rows ? rows[r] : r;
        std::vector<int64_t> s(nchans);          // this trial's row of the delay table
        for (int c = 0; c < nchans; ++c) s[c] = oracle_shift(dm_list[d], c, fch1, foff, tsamp);
        for (int64_t t = 0; t < nsamp; ++t) {
            double acc = 0.0, absacc = 0.0;
            for (int c = 0; c < nchans; ++c) {
                double x = (double)X[(size_t)c * in_stride + t + s[c]];
                acc += x;
                absacc += std::fabs(x);
            }
            D[(size_t)r * nsamp + t] = acc;
            if (A) A[(size_t)r * nsamp + t] = absacc;
        }
    }
}

// uint8 input.  The double sum is an exact integer (<= 255*nchans << 2^53);
// it is returned as int64 so the caller can check the int32 range itself.
void oracle_dedisperse_u8(const uint8_t* X, int nchans, int64_t nsamp, int64_t in_stride,
                          double fch1, double foff, double tsamp,
                          const double* dm_list, int ndm,
                          const int* rows, int nrows,
                          int64_t* D)
{
    int nr = rows ? nrows : ndm;
#pragma omp parallel for schedule(dynamic, 1)
    for (int r = 0; r < nr; ++r) {
        int d = rows ? rows[r] : r;
        std::vector<int64_t> s(nchans);          // this trial's row of the delay table
        for (int c = 0; c < nchans; ++c) s[c] = oracle_shift(dm_list[d], c, fch1, foff, tsamp);
        for (int64_t t = 0; t < nsamp; ++t) {
            double acc = 0.0;
            for (int c = 0; c < nchans; ++c)
                acc += (double)X[(size_t)c * in_stride + t + s[c]];
            D[(size_t)r * nsamp + t] = (int64_t)acc;
        }
    }
}

// Single elements (d_idx[i], t_idx[i]) -- for sampled parity on the big configs.
void oracle_elements_f32(const float* X, int nchans, int64_t in_stride,
                         double fch1, double foff, double tsamp, const double* dm_list,
                         const int* d_idx, const int64_t* t_idx, int64_t n,
                         double* D, double* A)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double acc = 0.0, absacc = 0.0;
        for (int c = 0; c < nchans; ++c) {
            int64_t s = oracle_shift(dm_list[d_idx[i]], c, fch1, foff, tsamp);
            double x = (double)X[(size_t)c * in_stride + t_idx[i] + s];
            acc += x;
            absacc += std::fabs(x);
        }
        D[i] = acc;
        if (A) A[i] = absacc;
    }
}

void oracle_elements_u8(const uint8_t* X, int nchans, int64_t in_stride,
                        double fch1, double foff, double tsamp, const double* dm_list,
                        const int* d_idx, const int64_t* t_idx, int64_t n, int64_t* D)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double acc = 0.0;
        for (int c = 0; c < nchans; ++c) {
            int64_t s = oracle_shift(dm_list[d_idx[i]], c, fch1, foff, tsamp);
            acc += (double)X[(size_t)c * in_stride + t_idx[i] + s];
        }
        D[i] = (int64_t)acc;
    }
}

// ---------------------------------------------------------------------------------------------
// Loop-interchanged variants: (d, c, t) with a per-trial row of double accumulators.  Every
// element D[d][t] still receives its channels in the order c = 0, 1, 2, ... into a double that
// starts at 0.0, so the results are BIT-IDENTICAL to the literal (d, t, c) nest above (a pin in
// tests/test_oracle_pins.py asserts exact equality on BASELINE.json configs 1-2 and on random
// small cases).  The inner loop streams over t, which the compiler vectorises: several times
// faster, so a whole-output pass over the largest configs is affordable.  The literal nest
// stays THE oracle and the timed CPU baseline; these exist for full-size parity passes and are
// reported separately in bench.py as "interchanged nest".
void oracle_dedisperse_f32_dct(const float* X, int nchans, int64_t nsamp, int64_t in_stride,
                               double fch1, double foff, double tsamp,
                               const double* dm_list, int ndm,
                               const int* rows, int nrows,
                               double* D, double* A)
{
    int nr = rows ? nrows : ndm;
#pragma omp parallel for schedule(dynamic, 1)
    for (int r = 0; r < nr; ++r) {
        int d = rows ? rows[r] : r;
        double* acc = D + (size_t)r * nsamp;
        double* absacc = A ? A + (size_t)r * nsamp : nullptr;
        for (int64_t t = 0; t < nsamp; ++t) acc[t] = 0.0;
        if (absacc)
            for (int64_t t = 0; t < nsamp; ++t) absacc[t] = 0.0;
        for (int c = 0; c < nchans; ++c) {
            const int64_t s = oracle_shift(dm_list[d], c, fch1, foff, tsamp);
            const float* x = X + (size_t)c * in_stride + s;
            for (int64_t t = 0; t < nsamp; ++t) acc[t] += (double)x[t];
            if (absacc)
                for (int64_t t = 0; t < nsamp; ++t) absacc[t] += std::fabs((double)x[t]);
        }
    }
}

void oracle_dedisperse_u8_dct(const uint8_t* X, int nchans, int64_t nsamp, int64_t in_stride,
                              double fch1, double foff, double tsamp,
                              const double* dm_list, int ndm,
                              const int* rows, int nrows,
                              int64_t* D)
{
    int nr = rows ? nrows : ndm;
#pragma omp parallel for schedule(dynamic, 1)
    for (int r = 0; r < nr; ++r) {
        int d = rows ? rows[r] : r;
        std::vector<double> acc((size_t)nsamp, 0.0);
        for (int c = 0; c < nchans; ++c) {
            const int64_t s = oracle_shift(dm_list[d], c, fch1, foff, tsamp);
            const uint8_t* x = X + (size_t)c * in_stride + s;
            for (int64_t t = 0; t < nsamp; ++t) acc[(size_t)t] += (double)x[t];
        }
        for (int64_t t = 0; t < nsamp; ++t) D[(size_t)r * nsamp + t] = (int64_t)acc[(size_t)t];
    }
}

}  // extern "C"
