// RFI mitigation front end on X (§3.3), in place on the
// device, before dedispersion.  Stages, in the paper's order (readings R20-R27):
//   1. averaged bandpass b_c = mean_t X[c][t]; least-squares polynomial of order p through it; RMSE of
//      the fit (§3.3.1);
//   2. channel thresholding (§3.3.2, eq 3.1): windows of W_c samples whose mean is off the fitted
//      bandpass value by more than T_c RMSE, and their two neighbours, are replaced by that value;
//   3. spectrum thresholding (§3.3.3, eq 3.2): spectra whose mean exceeds mu + T_s sigma of the spectrum
//      means lose the excess of their mean over the bandpass mean;
//   4. the fitted bandpass is subtracted from every spectrum.
//
// The thesis copies the averaged bandpass to the host, fits it there and runs one kernel per step
// with a write pass each.  Here everything stays on the device (the fit is one block solving the
// normal equations in a Legendre basis in double precision) and the replacements are never written as
// such: the window flags and the spectrum excesses are small side arrays, applied when the single
// output pass subtracts the bandpass.  Passes over X, plain form: two reads (window sums -- from which both
// the averaged bandpass and the window means follow -- and the spectrum means of the clipped data) and one
// read + write.  Fused form (16-byte aligned rows, window a multiple of 4 and <= 512): the first pass also
// leaves the column sums of tiles of 8-64 channels, the spectrum means come from those and from X at the
// replaced (channel, window) pairs only: one read and one read + write -- all HBM-bound streaming kernels.
// All means, the fit and the threshold comparisons are evaluated in double precision; the output is rounded
// once, from double, to float32.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>

#include "dd_internal.h"

namespace dd {

namespace {

constexpr int kThreads = 256;
constexpr int kMaxOrder = 12;
constexpr int kFitEntries = (kMaxOrder + 1) * (kMaxOrder + 4) / 2;   // entries of the augmented normal equations, upper triangle

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double block_sum(double v, double* red)
{
    v = warp_sum(v);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < kThreads / 32; ++w) s += red[w];
    return s;
}

// 1a. wsum[row][k] = sum of window k of channel row (one warp per window): the ONLY pass over X before the
// flags are known -- the averaged bandpass and the window means of stage 2 both follow from these sums.
__global__ void __launch_bounds__(kThreads)
dd_rfi_window_sums_kernel(const float* __restrict__ X, int nchans, int64_t n, int64_t stride, int64_t beam_stride,
                          int window, int nwin, double* __restrict__ wsum)
{
    const unsigned urow = blockIdx.y, ubeam = urow / (unsigned)nchans;       // 32-bit index arithmetic
    const int64_t row = urow;
    const int k = blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (k >= nwin) return;
    const float* x = X + (int64_t)ubeam * beam_stride + (int64_t)(urow - ubeam * (unsigned)nchans) * stride;
    const int64_t a = (int64_t)k * window, e = min(n, a + window);
    double s = 0.0;
    if ((window & 3) == 0 && e - a == window && (((uintptr_t)(x + a)) & 15) == 0) {
        const float4* x4 = reinterpret_cast<const float4*>(x + a);
        for (int i = lane; i < window / 4; i += 32) {
            const float4 v = __ldg(x4 + i);
            s += ((double)v.x + (double)v.y) + ((double)v.z + (double)v.w);
        }
    } else {
        for (int64_t t = a + lane; t < e; t += 32) s += (double)__ldg(x + t);
    }
    s = warp_sum(s);
    if (lane == 0) wsum[row * nwin + k] = s;
}

// 1a (fused form).  A warp takes window k of C consecutive channels: besides the window sums (same lanes, same
// order as above: identical values) every lane keeps the sums over those C channels of its 16 samples, and the
// warp leaves them in colpart[beam][channel tile][t] -- the spectrum means of stage 3 then need X only in the few
// windows where a channel is replaced.  For 16-byte aligned rows and window % 4 == 0, window <= 512.
// Rows are staged through a per-warp ring of kRing rows in shared memory with cp.async (16 bytes per lane and copy):
// three rows of every warp are in flight while it works on a fourth -- with plain loads the kernel held one row
// per warp in flight and ran at 4.7 TB/s (80 registers: 24 warps per SM).
constexpr int kRing = 4;
constexpr int kFusedSmem = (kThreads / 32) * kRing * 128 * 16;         // 8 warps x 4 rows x 2 KB

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem)
{
    const uint32_t sa = (uint32_t)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__global__ void __launch_bounds__(kThreads)
dd_rfi_window_col_sums_kernel(const float* __restrict__ X, int nchans, int64_t n, int64_t stride, int64_t beam_stride,
                              int window, int nwin, int C, int ntiles, int64_t np, double* __restrict__ wsum,
                              double* __restrict__ colpart)
{
    extern __shared__ float4 ring_all[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int k = blockIdx.x * (kThreads / 32) + warp;
    if (k >= nwin) return;
    float4* ring = ring_all + warp * (kRing * 128);
    const unsigned tile = blockIdx.y, ubeam = tile / (unsigned)ntiles, ct = tile - ubeam * (unsigned)ntiles;
    const int c0 = (int)ct * C;
    const int64_t a = (int64_t)k * window;
    const int len = (int)min((int64_t)window, n - a);                 // the last window may be shorter
    const float* x = X + (int64_t)ubeam * beam_stride + (int64_t)c0 * stride + a;
    double* ws = wsum + ((int64_t)ubeam * nchans + c0) * nwin + k;
    double col[4][4];
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int e = 0; e < 4; ++e) col[j][e] = 0.0;
    const int nfull = len >> 2;                                        // whole float4 groups of the window
    auto issue = [&](int c) {                                          // row c of the tile -> slot c % kRing (own lanes only)
        if (c < C) {
            const float* xr = x + (int64_t)c * stride;
            float4* slot = ring + (c % kRing) * 128;
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (lane + 32 * j < nfull) cp_async16(slot + lane + 32 * j, xr + 4 * (lane + 32 * j));
        }
        cp_async_commit();                                             // (an empty group keeps the count uniform)
    };
#pragma unroll
    for (int c = 0; c < kRing - 1; ++c) issue(c);
#pragma unroll 1
    for (int c = 0; c < C; ++c, ws += nwin) {
        issue(c + kRing - 1);
        cp_async_wait<kRing - 1>();                                    // row c has landed (every lane reads its own copies)
        const float4* slot = ring + (c % kRing) * 128;
        const float* xr = x + (int64_t)c * stride;
        double s = 0.0;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int i = lane + 32 * j;
            float4 v = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            if (i < nfull) {
                v = slot[i];
            } else if (4 * i < len) {                                  // the window's last, partial group
                v.x = __ldg(xr + 4 * i);
                if (4 * i + 1 < len) v.y = __ldg(xr + 4 * i + 1);
                if (4 * i + 2 < len) v.z = __ldg(xr + 4 * i + 2);
            }
            const double dx = (double)v.x, dy = (double)v.y, dz = (double)v.z, dw = (double)v.w;
            if (4 * i < window) s += (dx + dy) + (dz + dw);
            col[j][0] += dx;
            col[j][1] += dy;
            col[j][2] += dz;
            col[j][3] += dw;
        }
        s = warp_sum(s);
        if (lane == 0) *ws = s;
    }
    double* cp = colpart + ((int64_t)ubeam * ntiles + ct) * np + a;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int i = lane + 32 * j;
        if (i < nfull) {
            reinterpret_cast<double2*>(cp + 4 * i)[0] = make_double2(col[j][0], col[j][1]);
            reinterpret_cast<double2*>(cp + 4 * i)[1] = make_double2(col[j][2], col[j][3]);
        } else if (4 * i < len) {
            cp[4 * i] = col[j][0];
            if (4 * i + 1 < len) cp[4 * i + 1] = col[j][1];
            if (4 * i + 2 < len) cp[4 * i + 2] = col[j][2];
        }
    }
}

// 1a'. b[row] = mean over time of channel row = (sum of its window sums) / n  (one warp per row, fixed order)
__global__ void __launch_bounds__(kThreads)
dd_rfi_bandpass_kernel(const double* __restrict__ wsum, int64_t nrows, int nwin, int64_t n, double* __restrict__ b)
{
    const int64_t row = (int64_t)blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (row >= nrows) return;
    double s = 0.0;
    for (int k = lane; k < nwin; k += 32) s += wsum[row * nwin + k];
    s = warp_sum(s);
    if (lane == 0) b[row] = s / (double)n;
}

// 1b. One block per beam: least-squares polynomial of order p through (x_c, b_c), x_c the channel index
// mapped onto [-1, 1], in the Legendre basis P_0..P_p (normal equations, Gaussian elimination with partial
// pivoting, double).  Writes the fitted values B and stats = (rmse, mean_c B_c).
__global__ void __launch_bounds__(kThreads)
dd_rfi_fit_kernel(const double* __restrict__ b, int nchans, int order, double* __restrict__ B,
                  double* __restrict__ stats)
{
    __shared__ double red[kThreads / 32];
    __shared__ double G[(kMaxOrder + 1) * (kMaxOrder + 2)];   // augmented [p+1][p+2]
    __shared__ double coef[kMaxOrder + 1];
    __shared__ double part[kFitEntries][kThreads / 32];
    __shared__ double rk[kMaxOrder + 1];                      // 1 / k of the Legendre recurrence
    if (threadIdx.x <= kMaxOrder) rk[threadIdx.x] = threadIdx.x ? 1.0 / (double)threadIdx.x : 0.0;
    __syncthreads();
    const int beam = blockIdx.x;
    const double* bb = b + (int64_t)beam * nchans;
    const int p = min(order, nchans - 1), np1 = p + 1;
    auto absc = [&](int c) { return nchans > 1 ? 2.0 * (double)c / (double)(nchans - 1) - 1.0 : 0.0; };
    auto legendre = [&](double x, double* P) {                // P[0..p]
        P[0] = 1.0;
        if (p >= 1) P[1] = x;
        for (int k = 2; k <= p; ++k) P[k] = ((2.0 * k - 1.0) * x * P[k - 1] - (k - 1.0) * P[k - 2]) * rk[k];
    };
    // all (p+1)(p+4)/2 entries (i, j >= i) of the augmented normal equations (j == np1: right-hand side) in ONE
    // sweep over the channels: the basis is evaluated once per channel, a thread keeps its partial sums of every
    // entry (local memory: L1), then one warp reduction per entry and one barrier (order 4: 121 -> 30 us; before,
    // one sweep and one block-wide reduction per entry)
    {
        const int ne = np1 * (np1 + 3) / 2;
        double acc[kFitEntries];
        for (int e = 0; e < ne; ++e) acc[e] = 0.0;
        for (int c = threadIdx.x; c < nchans; c += kThreads) {
            double P[kMaxOrder + 1];
            legendre(absc(c), P);
            const double bc = bb[c];
            int e = 0;
            for (int i = 0; i < np1; ++i) {
                for (int j = i; j < np1; ++j) acc[e++] += P[i] * P[j];
                acc[e++] += P[i] * bc;
            }
        }
        const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
        for (int e = 0; e < ne; ++e) {
            const double s = warp_sum(acc[e]);
            if (lane == 0) part[e][warp] = s;
        }
        __syncthreads();
        if (threadIdx.x < ne) {
            double s = 0.0;
#pragma unroll
            for (int w = 0; w < kThreads / 32; ++w) s += part[threadIdx.x][w];
            int i = 0, j = threadIdx.x;                        // entry number -> (i, j)
            while (j > np1 - i) {
                j -= np1 - i + 1;
                ++i;
            }
            j += i;
            G[i * (np1 + 1) + j] = s;
            if (j < np1) G[j * (np1 + 1) + i] = s;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const int ld = np1 + 1;
        for (int k = 0; k < np1; ++k) {
            int piv = k;
            for (int r = k + 1; r < np1; ++r)
                if (fabs(G[r * ld + k]) > fabs(G[piv * ld + k])) piv = r;
            if (piv != k)
                for (int j = 0; j < ld; ++j) {
                    const double tmp = G[k * ld + j];
                    G[k * ld + j] = G[piv * ld + j];
                    G[piv * ld + j] = tmp;
                }
            const double d = G[k * ld + k];
            for (int r = k + 1; r < np1; ++r) {
                const double f = d != 0.0 ? G[r * ld + k] / d : 0.0;
                for (int j = k; j < ld; ++j) G[r * ld + j] -= f * G[k * ld + j];
            }
        }
        for (int k = np1 - 1; k >= 0; --k) {
            double s = G[k * ld + np1];
            for (int j = k + 1; j < np1; ++j) s -= G[k * ld + j] * coef[j];
            coef[k] = G[k * ld + k] != 0.0 ? s / G[k * ld + k] : 0.0;
        }
    }
    __syncthreads();
    double se = 0.0, sb = 0.0;
    for (int c = threadIdx.x; c < nchans; c += kThreads) {
        double P[kMaxOrder + 1];
        legendre(absc(c), P);
        double v = 0.0;
        for (int k = 0; k <= p; ++k) v += coef[k] * P[k];
        B[(int64_t)beam * nchans + c] = v;
        se += (bb[c] - v) * (bb[c] - v);
        sb += v;
    }
    se = block_sum(se, red);
    sb = block_sum(sb, red);
    if (threadIdx.x == 0) {
        stats[beam * 4 + 0] = sqrt(se / (double)nchans);      // RMSE (R22)
        stats[beam * 4 + 1] = sb / (double)nchans;            // mean of the fitted bandpass
    }
}

// 2. flag[row][k] = own[k-1] | own[k] | own[k+1],  own[k] = |mean of window k - B_row| > T_c * RMSE
// ("neighbouring blocks are also flagged", R24); the last, shorter window counts with its own length (R23).
__global__ void __launch_bounds__(kThreads)
dd_rfi_flags_kernel(const double* __restrict__ wsum, int64_t nrows, int nchans, int nwin, int window, int64_t n,
                    const double* __restrict__ B, const double* __restrict__ stats, double t_chan,
                    uint8_t* __restrict__ flag, uint8_t* __restrict__ chan_flags, uint8_t* __restrict__ dirty)
{
    const int64_t total = nrows * nwin;
    for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < total; i += (int64_t)gridDim.x * kThreads) {
        const int64_t row = i / nwin;
        const int k = (int)(i % nwin);
        const double Bc = B[row], level = t_chan * stats[(row / nchans) * 4 + 0];
        auto own = [&](int kk) {
            const int64_t a = (int64_t)kk * window, e = min(n, a + window);
            return fabs(wsum[row * nwin + kk] / (double)(e - a) - Bc) > level;
        };
        const bool f = own(k) || (k > 0 && own(k - 1)) || (k + 1 < nwin && own(k + 1));
        flag[i] = f;
        if (chan_flags) chan_flags[i] = f;
        if (f) dirty[(row / nchans) * nwin + k] = 1;       // some channel of this beam is replaced in window k
    }
}

constexpr int kSpecT = 128;                   // spectra per block of the spectrum-mean kernel
constexpr int kSpecQ = kThreads * 4 / kSpecT; // channel slices per block (threads = kSpecT x kSpecQ)

// 2'. (fused form) per beam, window with replaced channels and channel slice of the spectrum kernel: the replaced
// channels of the slice, ascending, in list[beam][k][c_lo(q) .. c_lo(q) + cnt[beam][k][q])  (one warp per window and
// slice; ballot compaction)
__global__ void __launch_bounds__(kThreads)
dd_rfi_flag_lists_kernel(const uint8_t* __restrict__ flag, const uint8_t* __restrict__ dirty, int nchans, int nwin,
                         uint16_t* __restrict__ list, int* __restrict__ cnt)
{
    const int w = blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5), lane = threadIdx.x & 31, beam = blockIdx.y;
    const int k = w / kSpecQ, q = w - k * kSpecQ;
    if (k >= nwin) return;
    const int cq = nchans / kSpecQ, c_lo = q * cq;                  // (the fused form needs nchans % kSpecQ == 0)
    int count = 0;
    if (dirty[(int64_t)beam * nwin + k]) {
        const uint8_t* fl = flag + (int64_t)beam * nchans * nwin + k;
        uint16_t* out = list + ((int64_t)beam * nwin + k) * nchans + c_lo;
        for (int c0 = c_lo; c0 < c_lo + cq; c0 += 32) {
            const int c = c0 + lane;
            const bool f = c < c_lo + cq && fl[(int64_t)c * nwin];
            const unsigned mask = __ballot_sync(0xffffffffu, f);
            if (f) out[count + __popc(mask & ((1u << lane) - 1u))] = (uint16_t)c;
            count += __popc(mask);
        }
    }
    if (lane == 0) cnt[((int64_t)beam * nwin + k) * kSpecQ + q] = count;
}

// 3a. m[beam][t] = mean over channels of the channel-clipped spectrum t.  Block = 128 spectra x 8 channel
// slices; a thread sums its slice's channels in ascending order (every load a coalesced row segment), the
// slices' partial sums meet in shared memory and are added in slice order.  Windows in which no channel of the
// beam is replaced (dirty[k] = 0: the usual case) skip the flag look-ups.  The block also leaves the sums of
// (m_t - bmean) and (m_t - bmean)^2 over its spectra in part[beam][block] (bmean = mean fitted bandpass: a
// shift close to the mean of the m_t), from which 3b forms mu and sigma.
__global__ void __launch_bounds__(kSpecT * kSpecQ)
dd_rfi_spectrum_kernel(const float* __restrict__ X, int nchans, int64_t n, int64_t stride, int64_t beam_stride,
                       int window, int nwin, const double* __restrict__ B, const uint8_t* __restrict__ flag,
                       const uint8_t* __restrict__ dirty, const double* __restrict__ stats, double* __restrict__ m,
                       double* __restrict__ part, const double* __restrict__ colpart, int C, int64_t np,
                       const uint16_t* __restrict__ list, const int* __restrict__ cnt)
{
    __shared__ double acc[kSpecQ][kSpecT];
    __shared__ double red[2][kSpecT / 32];
    const int beam = blockIdx.y, tx = threadIdx.x, q = threadIdx.y;
    const int64_t t = (int64_t)blockIdx.x * kSpecT + tx;
    const int64_t tc = min(t, n - 1);
    const int k = (int)((unsigned)tc / (unsigned)window);
    const float* x = X + (int64_t)beam * beam_stride + tc;
    const uint8_t* fl = flag + (int64_t)beam * nchans * nwin + k;
    const double* Bb = B + (int64_t)beam * nchans;
    const int cq = (nchans + kSpecQ - 1) / kSpecQ;
    const int c_lo = min(nchans, q * cq), c_hi = min(nchans, c_lo + cq);
    double s = 0.0;
    int c = c_lo;
    if (colpart) {
        // the first pass left the sums over tiles of C channels (slices are whole tiles); in a window where channels
        // are replaced, each of them contributes B_c instead of its sample: X is read at those (channel, window)
        // pairs only, taken from the slice's list of the window
        const double* cp = colpart + ((int64_t)beam * (nchans / C) + c_lo / C) * np + tc;
        for (int cc = c_lo; cc < c_hi; cc += C, cp += np) s += *cp;
        const int ne = cnt[((int64_t)beam * nwin + k) * kSpecQ + q];
        const uint16_t* le = list + ((int64_t)beam * nwin + k) * nchans + c_lo;
        for (int e = 0; e < ne; ++e) {
            const int cf = le[e];
            s += Bb[cf] - (double)__ldg(x + (int64_t)cf * stride);
        }
    } else if (!dirty[(int64_t)beam * nwin + k]) {
        for (; c + 8 <= c_hi; c += 8) {
            float v[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) v[j] = __ldg(x + (int64_t)(c + j) * stride);
#pragma unroll
            for (int j = 0; j < 8; ++j) s += (double)v[j];
        }
        for (; c < c_hi; ++c) s += (double)__ldg(x + (int64_t)c * stride);
    } else {
        for (; c + 8 <= c_hi; c += 8) {
            float v[8];
            uint8_t f[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                v[j] = __ldg(x + (int64_t)(c + j) * stride);
                f[j] = __ldg(fl + (int64_t)(c + j) * nwin);
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) s += f[j] ? Bb[c + j] : (double)v[j];
        }
        for (; c < c_hi; ++c) s += __ldg(fl + (int64_t)c * nwin) ? Bb[c] : (double)__ldg(x + (int64_t)c * stride);
    }
    acc[q][tx] = s;
    __syncthreads();
    if (q == 0) {
        double d1 = 0.0, d2 = 0.0;
        if (t < n) {
            double tot = acc[0][tx];
#pragma unroll
            for (int j = 1; j < kSpecQ; ++j) tot += acc[j][tx];
            tot /= (double)nchans;
            m[(int64_t)beam * n + t] = tot;
            d1 = tot - stats[beam * 4 + 1];
            d2 = d1 * d1;
        }
        d1 = warp_sum(d1);
        d2 = warp_sum(d2);
        if ((tx & 31) == 0) {
            red[0][tx >> 5] = d1;
            red[1][tx >> 5] = d2;
        }
    }
    __syncthreads();
    if (q == 0 && tx == 0) {
        double s1 = 0.0, s2 = 0.0;
#pragma unroll
        for (int w = 0; w < kSpecT / 32; ++w) {
            s1 += red[0][w];
            s2 += red[1][w];
        }
        part[((int64_t)beam * gridDim.x + blockIdx.x) * 2 + 0] = s1;
        part[((int64_t)beam * gridDim.x + blockIdx.x) * 2 + 1] = s2;
    }
}

// 3b. stats[beam][2..3] = mean and population standard deviation over time of m, from the blocks' partial
// sums about bmean (one block per beam, fixed order):  mu = bmean + S1 / n,  sigma^2 = S2 / n - (S1 / n)^2
__global__ void __launch_bounds__(kThreads)
dd_rfi_spectrum_stats_kernel(const double* __restrict__ part, int nblocks, int64_t n, double* __restrict__ stats)
{
    __shared__ double red[kThreads / 32];
    const int beam = blockIdx.x;
    const double* pp = part + (int64_t)beam * nblocks * 2;
    double s1 = 0.0, s2 = 0.0;
    for (int i = threadIdx.x; i < nblocks; i += kThreads) {
        s1 += pp[2 * i];
        s2 += pp[2 * i + 1];
    }
    s1 = block_sum(s1, red);
    s2 = block_sum(s2, red);
    if (threadIdx.x == 0) {
        const double d = s1 / (double)n;
        const double var = s2 / (double)n - d * d;
        stats[beam * 4 + 2] = stats[beam * 4 + 1] + d;
        stats[beam * 4 + 3] = var > 0.0 ? sqrt(var) : 0.0;
    }
}

// 3c. per spectrum: excess[t] = m_t - mean_c B_c if the spectrum is flagged (m_t - mu > T_s sigma), else 0;
// any4[t / 4] = some spectrum of the group of four is flagged (lets the write pass skip the excesses)
__global__ void __launch_bounds__(kThreads)
dd_rfi_excess_kernel(const double* __restrict__ m, int64_t n, const double* __restrict__ stats, double t_spec,
                     double* __restrict__ excess, uint8_t* __restrict__ any4, uint8_t* __restrict__ spec_flags)
{
    const int beam = blockIdx.y;
    const int64_t g = (int64_t)blockIdx.x * kThreads + threadIdx.x, t0 = 4 * g;
    if (t0 >= n) return;
    const double mu = stats[beam * 4 + 2], level = t_spec * stats[beam * 4 + 3], bmean = stats[beam * 4 + 1];
    bool any = false;
    for (int e = 0; e < 4 && t0 + e < n; ++e) {
        const double me = m[(int64_t)beam * n + t0 + e];
        const bool sf = (me - mu) > level;
        excess[(int64_t)beam * n + t0 + e] = sf ? me - bmean : 0.0;
        if (spec_flags) spec_flags[(int64_t)beam * n + t0 + e] = sf;
        any = any || sf;
    }
    any4[(int64_t)beam * ((n + 3) / 4) + g] = any;
}

// t / d for 0 <= t < 2^31 as a multiply and a shift: mul = ceil(2^(31+l) / d), shift = 31 + l, l = ceil(log2 d)
// (exact: the error term t e / 2^(31+l), e = mul d - 2^(31+l) < 2^l, stays below 1 / d)
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

struct FastDiv { uint32_t mul, shift; };
__device__ __forceinline__ uint32_t fast_div(uint32_t t, FastDiv f)
{
    return (uint32_t)(((uint64_t)t * f.mul) >> f.shift);
}

constexpr int kApplyJ = 8;                     // block steps per thread of the write pass (amortises the row set-up)

// 4. the single write pass: channel replacement, spectrum excess, bandpass subtraction; four consecutive
// samples per thread and step (16-byte accesses when the row allows); every value is formed in double and
// rounded once
__global__ void __launch_bounds__(kThreads)
dd_rfi_apply_kernel(float* __restrict__ X, int nchans, int64_t n, int64_t stride, int64_t beam_stride, int window,
                    int nwin, FastDiv div_window, const double* __restrict__ B, const uint8_t* __restrict__ flag,
                    const double* __restrict__ excess, const uint8_t* __restrict__ any4)
{
    const unsigned urow = blockIdx.y, ubeam = urow / (unsigned)nchans;       // 32-bit index arithmetic
    const int64_t row = urow;
    float* xrow = X + (int64_t)ubeam * beam_stride + (int64_t)(urow - ubeam * (unsigned)nchans) * stride;
    const double Bc = B[row];
    const uint8_t* fl = flag + row * nwin;
    const double* exb = excess + (int64_t)ubeam * n;
    const uint8_t* anyb = any4 + (int64_t)ubeam * ((n + 3) / 4);
    const unsigned uw = (unsigned)window;
#pragma unroll 1
    for (int j = 0; j < kApplyJ; ++j) {
        const int64_t g = ((int64_t)blockIdx.x * kApplyJ + j) * kThreads + threadIdx.x, t0 = 4 * g;
        if (t0 >= n) return;
        float* x = xrow + t0;
        // one 16-byte load per thread and step: ask L2 for the step after next (with eight steps: 1.50 -> 1.33 ms)
        if (j + 2 < kApplyJ && t0 + 2 * 4 * kThreads < n) prefetch_l2(x + 2 * 4 * kThreads);
        // window flags of the four samples (nsamp < 2^31 is checked by the host)
        const unsigned ut0 = (unsigned)t0;
        bool cf[4];
        if (window >= 4) {                                  // at most one window boundary inside the four samples
            const unsigned k0 = fast_div(ut0, div_window), next = (k0 + 1) * uw - ut0;   // samples left in window k0
            const bool cf0 = fl[k0], cf1 = next < 4 && k0 + 1 < (unsigned)nwin ? (bool)fl[k0 + 1] : cf0;
#pragma unroll
            for (int e = 0; e < 4; ++e) cf[e] = (unsigned)e >= next ? cf1 : cf0;
        } else {
#pragma unroll
            for (int e = 0; e < 4; ++e) cf[e] = fl[min(fast_div(ut0 + e, div_window), (unsigned)nwin - 1)];
        }
        const bool vec = t0 + 4 <= n && ((((uintptr_t)x) & 15) == 0);
        float v[4];
        if (vec) {
            const float4 q = *reinterpret_cast<const float4*>(x);
            v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
        } else {
#pragma unroll
            for (int e = 0; e < 4; ++e) v[e] = t0 + e < n ? x[e] : 0.0f;
        }
        double ex[4] = {0.0, 0.0, 0.0, 0.0};
        if (anyb[g]) {
#pragma unroll
            for (int e = 0; e < 4; ++e)
                if (t0 + e < n) ex[e] = exb[t0 + e];
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const double val = (cf[e] ? Bc : (double)v[e]) - ex[e];
            v[e] = (float)(val - Bc);
        }
        if (vec) {
            *reinterpret_cast<float4*>(x) = make_float4(v[0], v[1], v[2], v[3]);
        } else {
#pragma unroll
            for (int e = 0; e < 4; ++e)
                if (t0 + e < n) x[e] = v[e];
        }
    }
}

}  // namespace

int rfi_mitigate(float* X, int nchans, int64_t nsamp, int64_t stride, int64_t beam_stride, int nbeams,
                 const dd_rfi_params* prm, double* bandpass, double* fit, double* stats_out, uint8_t* chan_flags,
                 uint8_t* spec_flags, void* cuda_stream)
{
    if (!prm) return fail(DD_ERR_BAD_ARG, "params is null");
    if (nchans < 1 || nsamp < 0 || nbeams < 1) return fail(DD_ERR_BAD_ARG, "bad nchans / nsamp / nbeams");
    if (prm->poly_order < 0 || prm->poly_order > kMaxOrder) return fail(DD_ERR_BAD_ARG, "poly_order must be 0..12");
    if (prm->window < 1) return fail(DD_ERR_BAD_ARG, "window must be >= 1");
    if (!(prm->t_chan >= 0.0f) || !(prm->t_spec >= 0.0f)) return fail(DD_ERR_BAD_ARG, "thresholds must be >= 0");
    if (nsamp == 0) return DD_OK;
    if (nsamp > 2147483647LL) return fail(DD_ERR_UNSUPPORTED, "nsamp must fit int32: split the call in time");
    if (!X) return fail(DD_ERR_BAD_ARG, "X is null");
    if (stride < nsamp) return fail(DD_ERR_BAD_ARG, "stride is shorter than nsamp");
    if (nbeams > 1 && beam_stride < (int64_t)nchans * stride) return fail(DD_ERR_BAD_ARG, "beam stride is shorter than a beam");
    const int64_t nrows = (int64_t)nbeams * nchans;
    const int64_t nwin64 = (nsamp + prm->window - 1) / prm->window;
    const int64_t ntile = (nsamp + 4 * kThreads * kApplyJ - 1) / (4 * kThreads * kApplyJ);
    const int64_t nspec = (nsamp + kSpecT - 1) / kSpecT;
    if (nrows > 65535 || nbeams > 65535 || nwin64 > 2147483647LL || nspec > 2147483647LL)
        return fail(DD_ERR_UNSUPPORTED, "more than 65535 channel rows in one call: split the call by beam");
    const int nwin = (int)nwin64;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (nbeams == 1) beam_stride = 0;
    // workspace (doubles): b [nrows], B [nrows], stats [nbeams][4], m and excess [nbeams][nsamp], wsum [nrows][nwin];
    // part [nbeams][nspec][2]; (bytes): flag [nrows][nwin], any4 [nbeams][ceil(nsamp / 4)], dirty [nbeams][nwin]
    const int64_t ng4 = (nsamp + 3) / 4;
    // fused first pass (window sums + column sums of tiles of C channels): 16-byte aligned rows, window % 4 == 0 and
    // <= 512, channel slices of the spectrum kernel made of whole tiles
    int C = 0;
    if ((prm->window & 3) == 0 && prm->window <= 512 && (stride & 3) == 0 && (beam_stride & 3) == 0 &&
        (((uintptr_t)X) & 15) == 0 && nchans % kSpecQ == 0)
        for (int c : {64, 32, 16, 8})
            if ((nchans / kSpecQ) % c == 0) {
                C = c;
                break;
            }
    const int ntiles = C ? nchans / C : 0;
    const int64_t np = (nsamp + 3) / 4 * 4;                            // pitch of a column-sum row
    const size_t ncol = (size_t)nbeams * ntiles * np;
    if ((int64_t)nbeams * ntiles > 65535) C = 0;
    const size_t nd = (C ? ncol : 0) + (size_t)nrows * 2 + (size_t)nbeams * 4 + (size_t)2 * nbeams * nsamp +
                      (size_t)nrows * nwin + (size_t)2 * nbeams * nspec;
    // fused form only: cnt int32 [nbeams][nwin][kSpecQ], list uint16 [nbeams][nwin][nchans]
    const size_t nlist = C ? (size_t)nbeams * nwin * kSpecQ * sizeof(int) + (size_t)nrows * nwin * sizeof(uint16_t) : 0;
    char* ws = nullptr;
    int rc = workspace_alloc((void**)&ws, nd * sizeof(double) + nlist + (size_t)nrows * nwin + (size_t)nbeams * ng4 +
                                              (size_t)nbeams * nwin, cuda_stream);
    if (rc != DD_OK) return rc;
    double* colpart = C ? (double*)ws : nullptr;
    double* b = (double*)ws + (C ? ncol : 0);
    double* B = b + nrows;
    double* stats = B + nrows;
    double* m = stats + (size_t)nbeams * 4;
    double* excess = m + (size_t)nbeams * nsamp;
    double* wsum = excess + (size_t)nbeams * nsamp;
    double* part = wsum + (size_t)nrows * nwin;
    int* cnt = (int*)(part + (size_t)2 * nbeams * nspec);
    uint16_t* list = (uint16_t*)(cnt + (C ? (size_t)nbeams * nwin * kSpecQ : 0));
    uint8_t* flag = (uint8_t*)cnt + nlist;
    uint8_t* any4 = flag + (size_t)nrows * nwin;
    uint8_t* dirty = any4 + (size_t)nbeams * ng4;
    if (cudaMemsetAsync(dirty, 0, (size_t)nbeams * nwin, st) != cudaSuccess) {
        cudaFreeAsync(ws, st);
        return fail(DD_ERR_CUDA, "RFI mitigation: clearing the workspace failed");
    }
    constexpr int kWPB = kThreads / 32;                    // warps per block
    if (C && ensure_dyn_smem((const void*)dd_rfi_window_col_sums_kernel, kFusedSmem) != DD_OK) {
        cudaFreeAsync(ws, st);
        return DD_ERR_CUDA;
    }
    if (C)
        dd_rfi_window_col_sums_kernel<<<dim3((unsigned)((nwin + kWPB - 1) / kWPB), (unsigned)(nbeams * ntiles)), kThreads,
                                        kFusedSmem, st>>>(X, nchans, nsamp, stride, beam_stride, prm->window, nwin, C, ntiles, np, wsum,
                                              colpart);
    else
        dd_rfi_window_sums_kernel<<<dim3((unsigned)((nwin + kWPB - 1) / kWPB), (unsigned)nrows), kThreads, 0, st>>>(
            X, nchans, nsamp, stride, beam_stride, prm->window, nwin, wsum);
    dd_rfi_bandpass_kernel<<<(unsigned)((nrows + kWPB - 1) / kWPB), kThreads, 0, st>>>(wsum, nrows, nwin, nsamp, b);
    dd_rfi_fit_kernel<<<(unsigned)nbeams, kThreads, 0, st>>>(b, nchans, prm->poly_order, B, stats);
    dd_rfi_flags_kernel<<<(unsigned)std::min<int64_t>((nrows * nwin + kThreads - 1) / kThreads, 4096), kThreads, 0, st>>>(
        wsum, nrows, nchans, nwin, prm->window, nsamp, B, stats, (double)prm->t_chan, flag, chan_flags, dirty);
    if (C)
        dd_rfi_flag_lists_kernel<<<dim3((unsigned)(((int64_t)nwin * kSpecQ + kWPB - 1) / kWPB), (unsigned)nbeams), kThreads, 0, st>>>(
            flag, dirty, nchans, nwin, list, cnt);
    dd_rfi_spectrum_kernel<<<dim3((unsigned)nspec, (unsigned)nbeams), dim3(kSpecT, kSpecQ), 0, st>>>(
        X, nchans, nsamp, stride, beam_stride, prm->window, nwin, B, flag, dirty, stats, m, part, colpart, C, np, list, cnt);
    dd_rfi_spectrum_stats_kernel<<<(unsigned)nbeams, kThreads, 0, st>>>(part, (int)nspec, nsamp, stats);
    dd_rfi_excess_kernel<<<dim3((unsigned)((ng4 + kThreads - 1) / kThreads), (unsigned)nbeams), kThreads, 0, st>>>(
        m, nsamp, stats, (double)prm->t_spec, excess, any4, spec_flags);
    FastDiv dw;
    {
        uint32_t l = 0;
        while ((1ull << l) < (uint64_t)prm->window) ++l;
        dw.shift = 31 + l;
        dw.mul = (uint32_t)(((1ull << dw.shift) + (uint64_t)prm->window - 1) / (uint64_t)prm->window);
    }
    dd_rfi_apply_kernel<<<dim3((unsigned)ntile, (unsigned)nrows), kThreads, 0, st>>>(
        X, nchans, nsamp, stride, beam_stride, prm->window, nwin, dw, B, flag, excess, any4);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && bandpass)
        e = cudaMemcpyAsync(bandpass, b, (size_t)nrows * sizeof(double), cudaMemcpyDeviceToDevice, st);
    if (e == cudaSuccess && fit)
        e = cudaMemcpyAsync(fit, B, (size_t)nrows * sizeof(double), cudaMemcpyDeviceToDevice, st);
    if (e == cudaSuccess && stats_out)
        e = cudaMemcpyAsync(stats_out, stats, (size_t)nbeams * 4 * sizeof(double), cudaMemcpyDeviceToDevice, st);
    cudaFreeAsync(ws, st);
    if (e != cudaSuccess) return fail(DD_ERR_CUDA, std::string("RFI mitigation: ") + cudaGetErrorString(e));
    return DD_OK;
}

}  // namespace dd
