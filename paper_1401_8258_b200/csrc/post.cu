// Post-processing of the dedispersed time series and first stage of event detection
// (§3.5-3.6), on the device, so that the (DM, t) plane
// -- 4 to 17 GB on the BASELINE.json workloads -- never has to cross PCIe: what leaves the GPU is
// the list of (beam, DM, time, S/N) candidates.
//
// Steps, in the paper's order (readings R15-R19):
//   1. windowed median, odd w <= 9 centred on the sample (eq 3.4), ends clamped;
//   2. least-squares line over the whole series subtracted (pass 1: regression
//      parameters, pass 2: subtraction + standard deviation);
//   3. division by that standard deviation (pass 3);
//   4. threshold at n sigma -> (time, DM, intensity) triplets per beam.
//
// Two kernels.  dd_post_stats_kernel: one block per series, ONE pass: sum u, sum (t - tm) u and
// sum u^2 of u = y - y_0 in double (the median is formed on the fly from the raw series, never
// stored); slope, intercept and the residual's standard deviation follow from the normal equations
// (the thesis' two passes give the same numbers; the offset y_0 keeps a constant series at sigma = 0
// exactly).  dd_post_apply_kernel: grid over (time tiles, series); every thread forms four
// consecutive medians from 4 + (w - 1) loaded samples, subtracts the line, scales, optionally stores
// the processed series (16-byte stores) and appends the samples above the threshold to the
// candidate list through an atomic cursor.  Candidates-only calls: the statistics pass also leaves the largest
// median of every 128-sample chunk and dd_post_scan_kernel reads D only in chunks that can hold a detection.
// HBM traffic: D is read once (candidates only) or twice and written at most once, against seven passes for
// the step-by-step pipeline of §3.5; the kernels are HBM-bound.
// The thesis used one kernel per step with the series staged in shared memory.
#include <cuda_runtime.h>

#include <cmath>
#include <mutex>
#include <type_traits>

#include "dd_internal.h"

namespace dd {

namespace {

constexpr int kThreads = 512;
constexpr int kPer = 4;                       // consecutive samples per thread
constexpr int kTile = kThreads * kPer;        // samples per block step


// min / max as single instructions (FMNMX / IMNMX); the series hold no NaN by contract (R14: not handled)
__device__ __forceinline__ float mn(float a, float b) { return fminf(a, b); }
__device__ __forceinline__ float mx(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ int32_t mn(int32_t a, int32_t b) { return min(a, b); }
__device__ __forceinline__ int32_t mx(int32_t a, int32_t b) { return max(a, b); }
template <typename T> __device__ __forceinline__ void cmpx(T& a, T& b)
{
    const T lo = mn(a, b), hi = mx(a, b);
    a = lo;
    b = hi;
}
// median of W values: selection only (the result is one of the inputs), static indices, branch-free.
// W = 3 and 5 use the short min / max forms (4 and 10 operations: the median of five is the median of
// the fifth value, the larger of the two pair minima and the smaller of the two pair maxima); W = 7 a
// 13-comparator selection network of which the compiler keeps the 20 min / max that reach v[3]; W = 9 three
// sorted triples (the median of nine is the median of: the largest minimum, the median of the middles, the
// smallest maximum; 30 operations).  Both checked on all 0/1 inputs (min / max networks: the 0-1 principle).
template <typename T> __device__ __forceinline__ T med3(T a, T b, T c) { return mx(mn(a, b), mn(mx(a, b), c)); }
template <typename T> __device__ __forceinline__ void sort3(T& a, T& b, T& c)
{
    cmpx(a, b);
    cmpx(b, c);
    cmpx(a, b);
}
// median of nine from three ascending triples
template <typename T> __device__ __forceinline__ T med9_sorted(const T (&p)[3], const T (&q)[3], const T (&r)[3])
{
    return med3(mx(mx(p[0], q[0]), r[0]), med3(p[1], q[1], r[1]), mn(mn(p[2], q[2]), r[2]));
}
template <typename T, int W> __device__ __forceinline__ T median_of(T (&v)[W])
{
    if constexpr (W == 3) {
        return med3(v[0], v[1], v[2]);
    } else if constexpr (W == 5) {
        const T lo = mx(mn(v[0], v[1]), mn(v[2], v[3])), hi = mn(mx(v[0], v[1]), mx(v[2], v[3]));
        return mx(mn(lo, hi), mn(mx(lo, hi), v[4]));
    } else if constexpr (W == 7) {
        cmpx(v[0], v[5]); cmpx(v[0], v[3]); cmpx(v[1], v[6]); cmpx(v[2], v[4]); cmpx(v[0], v[1]);
        cmpx(v[3], v[5]); cmpx(v[2], v[6]); cmpx(v[2], v[3]); cmpx(v[3], v[6]); cmpx(v[4], v[5]);
        cmpx(v[1], v[4]); cmpx(v[1], v[3]); cmpx(v[3], v[4]);
        return v[3];
    } else if constexpr (W == 9) {
        T t[3][3];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            t[i][0] = v[3 * i], t[i][1] = v[3 * i + 1], t[i][2] = v[3 * i + 2];
            sort3(t[i][0], t[i][1], t[i][2]);
        }
        return med9_sorted(t[0], t[1], t[2]);
    } else {
#pragma unroll
        for (int round = 0; round < W; ++round)
#pragma unroll
            for (int i = round & 1; i + 1 < W; i += 2) cmpx(v[i], v[i + 1]);
        return v[W / 2];
    }
}

// The kPer medians of samples t0 .. t0+kPer-1 of one series; window indices clamped to
// [0, n-1] (R15).  Samples past the end give the clamped windows' medians (never used).
// n < 2^31 (checked by the caller): 32-bit sample indices.
template <typename T, int W>
__device__ __forceinline__ void medians4(const T* __restrict__ row, unsigned t0, unsigned n, T (&m)[kPer],
                                         bool row_aligned)   // row is 16-byte aligned (t0 is a multiple of 4)
{
    constexpr int H = (W - 1) / 2;
    T x[kPer + 2 * H];
    static_assert(sizeof(T) == 4 && kPer == 4 && H <= 4, "the aligned path loads three 16-byte vectors");
    if (row_aligned && t0 >= 4 && t0 + 8 <= n) {
        // interior, 16-byte aligned: the thread's four samples and the aligned vectors on either side
        // (the neighbours' own samples: L1 hits) instead of 4 + 2 H scalar loads
        const int4* src = reinterpret_cast<const int4*>(row + t0);
        const int4 l = __ldg(src - 1), c = __ldg(src), r = __ldg(src + 1);
        const int w12[12] = {l.x, l.y, l.z, l.w, c.x, c.y, c.z, c.w, r.x, r.y, r.z, r.w};
#pragma unroll
        for (int i = 0; i < kPer + 2 * H; ++i) {
            union { int i; T t; } u;
            u.i = w12[4 - H + i];
            x[i] = u.t;
        }
    } else if (t0 >= H && t0 + kPer + H <= n) {           // interior: no clamping
        const T* src = row + (t0 - H);
#pragma unroll
        for (int i = 0; i < kPer + 2 * H; ++i) x[i] = __ldg(src + i);
    } else {
#pragma unroll
        for (int i = 0; i < kPer + 2 * H; ++i) {
            int64_t j = (int64_t)t0 - H + i;
            j = j < 0 ? 0 : (j > (int64_t)n - 1 ? (int64_t)n - 1 : j);
            x[i] = __ldg(row + j);
        }
    }
    if constexpr (W == 5) {
        // two adjacent windows share four values: with b <= c the middle two of the shared four, the median of
        // the four and a fifth value e is e clamped to [b, c] -- 12 min / max operations per two medians
#pragma unroll
        for (int e = 0; e < kPer; e += 2) {
            const T p0 = mn(x[e + 1], x[e + 2]), p1 = mx(x[e + 1], x[e + 2]);
            const T q0 = mn(x[e + 3], x[e + 4]), q1 = mx(x[e + 3], x[e + 4]);
            const T u = mx(p0, q0), v = mn(p1, q1);            // the middle two, in either order
            const T b = mn(u, v), c = mx(u, v);
            m[e] = mn(mx(x[e], b), c);
            m[e + 1] = mn(mx(x[e + 5], b), c);
        }
    } else if constexpr (W == 9) {
        // window e is the triples starting at e, e + 3, e + 6: the four windows need ten sorted triples, not twelve
        T t[10][3];
#pragma unroll
        for (int i = 0; i < 10; ++i) {
            t[i][0] = x[i], t[i][1] = x[i + 1], t[i][2] = x[i + 2];
            sort3(t[i][0], t[i][1], t[i][2]);
        }
#pragma unroll
        for (int e = 0; e < kPer; ++e) m[e] = med9_sorted(t[e], t[e + 3], t[e + 6]);
    } else {
#pragma unroll
        for (int e = 0; e < kPer; ++e) {
            T v[W];
#pragma unroll
            for (int i = 0; i < W; ++i) v[i] = x[e + i];
            m[e] = median_of<T, W>(v);
        }
    }
}

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// chunk maxima are kept as signed integer keys: the value itself for int32 series, the order-preserving map of the
// bit pattern for float32 series (its own inverse), so that the warp maximum is one REDUX
__device__ __forceinline__ int32_t max_key(int32_t v) { return v; }
__device__ __forceinline__ int32_t max_key(float v)
{
    const int32_t b = __float_as_int(v);
    return b ^ ((b >> 31) & 0x7fffffff);
}
template <typename T> __device__ __forceinline__ float key_to_float_up(int32_t k)      // never below the value
{
    if constexpr (std::is_integral<T>::value) return __int2float_ru(k);
    else return __int_as_float(k ^ ((k >> 31) & 0x7fffffff));
}
template <typename T> __device__ __forceinline__ T lowest_of();
template <> __device__ __forceinline__ float lowest_of<float>() { return -INFINITY; }
template <> __device__ __forceinline__ int32_t lowest_of<int32_t>() { return INT32_MIN; }

constexpr int kChunk = 32 * kPer;             // samples of one warp step: the granularity of the chunk maxima

__device__ __forceinline__ double block_sum(double v, double* red)
{
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();                                      // red may still be read from the previous reduction
    if (lane == 0) red[warp] = v;
    __syncthreads();
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < kThreads / 32; ++w) s += red[w];  // same order in every thread
    return s;
}

// stats[row] = (intercept, slope, sigma): least-squares line through (t, y_t), t = 0..n-1, of the
// median-filtered series and the population standard deviation of the residual, from ONE pass:
// with u_t = y_t - y_0 (the offset removes the level, so a constant series gives exact zeros) and
// tc = t - (n-1)/2,  slope = sum tc u / sum tc^2,  mean = y_0 + sum u / n,
// SS_res = sum u^2 - (sum u)^2 / n - slope^2 sum tc^2  (the normal equations' residual), all in double.
template <typename T, int W, bool CM>
__global__ void __launch_bounds__(kThreads)
dd_post_stats_kernel(const T* __restrict__ D, int64_t stride, int64_t beam_stride, int ndm, int64_t n,
                     double* __restrict__ stats, int32_t* __restrict__ cmax)
{
    __shared__ double red[kThreads / 32];
    const int64_t r = blockIdx.x;
    const T* row = D + (r / ndm) * beam_stride + (r % ndm) * stride;
    const double tm = 0.5 * (double)(n - 1);
    const unsigned n32 = (unsigned)n;
    T first[kPer];
    const bool row_aligned = ((uintptr_t)row & 15) == 0;
    medians4<T, W>(row, 0u, n32, first, row_aligned);
    const double y0 = (double)first[0];
    double su = 0.0, stu = 0.0, suu = 0.0;
    double tc0 = (double)(threadIdx.x * kPer) - tm;       // t0 - tm as a running double (exact: multiples of 1/2)
    // cmax (optional): the largest median of every chunk of 128 samples (one warp step), which lets a
    // candidates-only second pass skip the chunks that cannot hold a detection.  The trip count is uniform over
    // a warp (warp-wide maximum); threads past the end form clamped medians that are not used.
    const unsigned lane4 = (threadIdx.x & 31) * kPer;
    int32_t* cmp = CM ? cmax + r * (int64_t)((n32 + kChunk - 1) / kChunk) + (threadIdx.x >> 5) : nullptr;   // this warp's first chunk
    for (unsigned t0 = threadIdx.x * kPer; t0 - (CM ? lane4 : 0u) < n32; t0 += kTile, tc0 += (double)kTile) {
        // one load group per thread and trip leaves too few bytes in flight (3 blocks x 512 threads x 16 bytes
        // per SM): ask L2 for the trip after next (no register cost; 1.01 -> 0.79 ms on config 3's plane)
        if (t0 + 2 * kTile < n32) prefetch_l2(row + t0 + 2 * kTile);
        T m[kPer];
        medians4<T, W>(row, t0, n32, m, row_aligned);
        if constexpr (CM) {
            T top;
            if (t0 + kPer <= n32) {
                top = mx(mx(m[0], m[1]), mx(m[2], m[3]));
            } else {
                top = lowest_of<T>();
#pragma unroll
                for (int e = 0; e < kPer; ++e)
                    if (t0 + e < n32) top = mx(top, m[e]);
            }
            const int32_t key = __reduce_max_sync(0xffffffffu, max_key(top));
            if (lane4 == 0) *cmp = key;
            cmp += kTile / kChunk;
        }
        double u[kPer];
#pragma unroll
        for (int e = 0; e < kPer; ++e) u[e] = (double)m[e] - y0;
        if (t0 + kPer <= n32) {
            // four samples at once: sum u, sum e u and sum u^2 of the group, then tc0 (sum u) + sum e u:
            // 16 double operations per four samples instead of 28 (the build has --fmad=false: the fused
            // multiply-adds here are explicit)
            const double s1 = (u[0] + u[1]) + (u[2] + u[3]);
            const double s2 = fma(3.0, u[3], fma(2.0, u[2], u[1]));
            const double q = fma(u[3], u[3], fma(u[2], u[2], fma(u[1], u[1], u[0] * u[0])));
            su += s1;
            stu = fma(tc0, s1, stu) + s2;
            suu += q;
        } else {
#pragma unroll
            for (int e = 0; e < kPer; ++e)
                if (t0 + e < n32) {
                    su += u[e];
                    stu = fma(tc0 + (double)e, u[e], stu);
                    suu = fma(u[e], u[e], suu);
                }
        }
    }
    su = block_sum(su, red);
    stu = block_sum(stu, red);
    suu = block_sum(suu, red);
    if (threadIdx.x == 0) {
        const double dn = (double)n;
        const double stt = dn * (dn * dn - 1.0) / 12.0;   // sum (t - tm)^2
        const double slope = stt > 0.0 ? stu / stt : 0.0;
        const double ss_tot = suu - su * su / dn;
        double ss = ss_tot - slope * slope * stt;
        // a series that is a straight line to rounding (ss / ss_tot ~ 1e-16) has no residual to normalise
        if (!(ss > 1e-24 * fmax(ss_tot, suu))) ss = 0.0;
        stats[r * 3 + 0] = y0 + su / dn - slope * tm;
        stats[r * 3 + 1] = slope;
        stats[r * 3 + 2] = sqrt(ss / dn);
    }
}

struct ApplyParams {
    int64_t stride, beam_stride, n;
    int ndm;
    unsigned ntiles, steps;                                // grid tiles per series, block steps per tile
    int detrend, normalise, threshold_on;
    double nsigma;
    const double* stats;
    int32_t* cmax;                                         // chunk maxima (keys) of the statistics pass, or null
    float* Z;
    int64_t z_stride, z_beam_stride;
    dd_candidate* cand;
    int64_t capacity;
    unsigned long long* count;
};

constexpr int kApplyJ = 16;                    // most block steps per thread of the apply kernel (long running prefetch, row set-up amortised)

template <typename T, int W>
__global__ void __launch_bounds__(kThreads)
dd_post_apply_kernel(const T* __restrict__ D, const ApplyParams p)
{
    const unsigned r = blockIdx.x / p.ntiles;             // time tiles fastest (1-D grid: no 65535 limit on series)
    const int beam = (int)(r / (unsigned)p.ndm), dm = (int)(r - (unsigned)beam * (unsigned)p.ndm);
    const T* row = D + (int64_t)beam * p.beam_stride + (int64_t)dm * p.stride;
    double intercept = 0.0, slope = 0.0, sigma = 0.0;
    if (p.detrend) {
        intercept = p.stats[(int64_t)r * 3 + 0];
        slope = p.stats[(int64_t)r * 3 + 1];
        sigma = p.stats[(int64_t)r * 3 + 2];
    }
    const double inv = sigma > 0.0 ? 1.0 / sigma : 0.0;    // sigma = 0: all-zero output (R17)
    float* zrow = p.Z ? p.Z + (int64_t)beam * p.z_beam_stride + (int64_t)dm * p.z_stride : nullptr;
    // Threshold-only calls (no series output) screen in single precision.  With sigma > 0 and n sigma >= 0 a
    // sample passes  (m - line(t)) / sigma > n sigma  only if  m > line(t) + n sigma * sigma - delta =: L(t),
    // delta <= 2^-48 S the rounding of the double evaluation, S = |slope| n + |intercept| + n sigma * sigma.
    // lo(t) = fl32(b t + a), a = intercept + n sigma * sigma - 2^-21 S rounded down, lies below L(t) for all
    // t < n (the float evaluation of the line is off by at most 2^-22 |slope| n + 2^-23 |a|).  Samples
    // above lo(t) -- a handful per series at 6 sigma -- take the double-precision decision below, so the
    // candidates are exactly those of the unscreened evaluation.
    const bool screen = !zrow && p.threshold_on && sigma > 0.0 && p.nsigma >= 0.0;
    float scr_a = 0.0f, scr_b = 0.0f;
    const unsigned n32 = (unsigned)p.n;
    if (screen) {
        const double level = p.nsigma * sigma;
        const double margin = 0x1p-21 * (fabs(slope) * (double)p.n + fabs(intercept) + level);
        scr_a = __double2float_rd(intercept + level - margin);
        scr_b = (float)slope;
    }
    const unsigned tile0 = (blockIdx.x - r * p.ntiles) * p.steps;
    {   // as in the statistics kernel: ask L2 for the next two steps, then for the step after next in every step
        const unsigned tp = (tile0 * kThreads + threadIdx.x) * kPer;
        if (p.steps > 1 && tp + kTile < n32) prefetch_l2(row + tp + kTile);
    }
#pragma unroll 1
    for (unsigned j = 0; j < p.steps; ++j) {
        const unsigned t0 = ((tile0 + j) * kThreads + threadIdx.x) * kPer;
        if (t0 >= n32) return;
        if (j + 2 < p.steps && t0 + 2 * kTile < n32) prefetch_l2(row + t0 + 2 * kTile);
        T m[kPer];
        medians4<T, W>(row, t0, n32, m, ((uintptr_t)(row + t0) & 15) == 0);
        if (screen) {
            const float tf = (float)t0;
            bool any = false;
#pragma unroll
            for (int e = 0; e < kPer; ++e) {
                float mf;
                if constexpr (std::is_integral<T>::value) mf = __int2float_ru((int)m[e]);   // never below m
                else mf = (float)m[e];
                any |= mf > fmaf(scr_b, tf + (float)e, scr_a);
            }
            if (!any) continue;
        }
        const double td0 = (double)t0;                     // exact; t0 + e as td0 + e is exact too
        float out[kPer];
#pragma unroll
        for (int e = 0; e < kPer; ++e) {
            double v = (double)m[e];
            if (p.detrend) v -= intercept + slope * (td0 + (double)e);
            // un-normalised series are compared against n * sigma; same decision, same precision
            const double snr = p.detrend ? v * inv : v;
            if (p.normalise) v = snr;
            out[e] = (float)v;
            if (p.threshold_on && t0 + e < n32 && snr > p.nsigma) {
                const unsigned long long at = atomicAdd(p.count, 1ull);
                if ((int64_t)at < p.capacity) {
                    dd_candidate c;
                    c.beam = beam;
                    c.dm = dm;
                    c.t = (int32_t)(t0 + e);
                    c.value = (float)snr;
                    p.cand[at] = c;
                }
            }
        }
        if (zrow) {
            float* z = zrow + t0;
            if (t0 + kPer <= n32 && (((uintptr_t)z) & 15) == 0) {
                *reinterpret_cast<float4*>(z) = make_float4(out[0], out[1], out[2], out[3]);
            } else {
#pragma unroll
                for (int e = 0; e < kPer; ++e)
                    if (t0 + e < n32) z[e] = out[e];
            }
        }
    }
}

// Candidates-only second pass when the statistics pass has left the chunk maxima: a lane tests one chunk of 128
// samples -- its largest median against lo at both ends of the chunk (L(t) = line(t) + n sigma * sigma is linear, so
// its minimum over the chunk is at an end, and lo < L there: see the screen of the apply kernel) -- and the warp then
// takes the chunks that can hold a detection one by one (medians again, double-precision decision for every
// sample).  D is read only where candidates are: 4 bytes of keys per 512 bytes of D otherwise.
template <typename T, int W>
__global__ void __launch_bounds__(kThreads)
dd_post_scan_kernel(const T* __restrict__ D, const ApplyParams p, unsigned blocks_per_row)
{
    const unsigned r = blockIdx.x / blocks_per_row;
    const int beam = (int)(r / (unsigned)p.ndm), dm = (int)(r - (unsigned)beam * (unsigned)p.ndm);
    const T* row = D + (int64_t)beam * p.beam_stride + (int64_t)dm * p.stride;
    const double intercept = p.stats[(int64_t)r * 3 + 0], slope = p.stats[(int64_t)r * 3 + 1];
    const double sigma = p.stats[(int64_t)r * 3 + 2];
    if (!(sigma > 0.0)) return;                            // sigma = 0: all-zero series, nothing above n sigma >= 0
    const bool row_aligned = ((uintptr_t)row & 15) == 0;
    const double inv = 1.0 / sigma;
    const double level = p.nsigma * sigma;
    const double margin = 0x1p-21 * (fabs(slope) * (double)p.n + fabs(intercept) + level);
    const float scr_a = __double2float_rd(intercept + level - margin), scr_b = (float)slope;
    const unsigned n32 = (unsigned)p.n, nchunk = (n32 + kChunk - 1) / kChunk;
    const int32_t* cmrow = p.cmax + (int64_t)r * nchunk;
    const unsigned lane = threadIdx.x & 31;
    const unsigned c = ((blockIdx.x - r * blocks_per_row) * (kThreads / 32) + (threadIdx.x >> 5)) * 32 + lane;
    bool hot = false;
    if (c < nchunk) {
        const float tf = (float)(c * kChunk);
        const float lo = fminf(fmaf(scr_b, tf, scr_a), fmaf(scr_b, tf + (float)(kChunk - 1), scr_a));
        hot = key_to_float_up<T>(cmrow[c]) > lo;
    }
    unsigned todo = __ballot_sync(0xffffffffu, hot);
    while (todo) {
        const unsigned ch = c - lane + (unsigned)(__ffs(todo) - 1);
        todo &= todo - 1;
        const unsigned t0 = ch * kChunk + lane * kPer;
        if (t0 >= n32) continue;
        T m[kPer];
        medians4<T, W>(row, t0, n32, m, row_aligned);
        const double td0 = (double)t0;
#pragma unroll
        for (int e = 0; e < kPer; ++e) {
            const double v = (double)m[e] - (intercept + slope * (td0 + (double)e));
            const double snr = v * inv;
            if (t0 + e < n32 && snr > p.nsigma) {
                const unsigned long long at = atomicAdd(p.count, 1ull);
                if ((int64_t)at < p.capacity) {
                    dd_candidate cd;
                    cd.beam = beam;
                    cd.dm = dm;
                    cd.t = (int32_t)(t0 + e);
                    cd.value = (float)snr;
                    p.cand[at] = cd;
                }
            }
        }
    }
}

template <typename T, int W>
int launch_w(const void* D, int64_t nrows, const ApplyParams& ap, double* stats, cudaStream_t st)
{
    if (ap.detrend && ap.cmax)
        dd_post_stats_kernel<T, W, true><<<(unsigned)nrows, kThreads, 0, st>>>(
            (const T*)D, ap.stride, ap.beam_stride, ap.ndm, ap.n, stats, ap.cmax);
    else if (ap.detrend)
        dd_post_stats_kernel<T, W, false><<<(unsigned)nrows, kThreads, 0, st>>>(
            (const T*)D, ap.stride, ap.beam_stride, ap.ndm, ap.n, stats, nullptr);
    if (ap.cmax) {                                         // candidates only, chunk maxima at hand
        const int64_t nchunk = (ap.n + kChunk - 1) / kChunk, per_block = (kThreads / 32) * 32;
        const unsigned bpr = (unsigned)((nchunk + per_block - 1) / per_block);
        dd_post_scan_kernel<T, W><<<(unsigned)(nrows * bpr), kThreads, 0, st>>>((const T*)D, ap, bpr);
    } else if (ap.Z || ap.threshold_on) {
        dd_post_apply_kernel<T, W><<<(unsigned)(nrows * ap.ntiles), kThreads, 0, st>>>((const T*)D, ap);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(DD_ERR_CUDA, std::string("post-processing launch: ") + cudaGetErrorString(e));
    return DD_OK;
}

template <typename T>
int launch_t(int w, const void* D, int64_t nrows, const ApplyParams& ap, double* stats, cudaStream_t st)
{
    switch (w) {
        case 1: return launch_w<T, 1>(D, nrows, ap, stats, st);
        case 3: return launch_w<T, 3>(D, nrows, ap, stats, st);
        case 5: return launch_w<T, 5>(D, nrows, ap, stats, st);
        case 7: return launch_w<T, 7>(D, nrows, ap, stats, st);
        case 9: return launch_w<T, 9>(D, nrows, ap, stats, st);
    }
    return fail(DD_ERR_BAD_ARG, "median_window must be 0, 1, 3, 5, 7 or 9");
}

}  // namespace

int post_launches(const dd_post_params* prm, bool want_series)
{
    return (prm->detrend ? 1 : 0) + ((want_series || prm->threshold_on) ? 1 : 0);
}

static int postprocess_impl(int dtype, const void* D, int64_t stride, int64_t beam_stride, int ndm, int64_t nsamp,
                            int nbeams, const dd_post_params* prm, float* Z, int64_t z_stride, int64_t z_beam_stride,
                            double* stats, dd_candidate* cand, int64_t capacity, unsigned long long* count,
                            void* cuda_stream, bool may_allocate)
{
    if (!prm) return fail(DD_ERR_BAD_ARG, "params is null");
    if (dtype != DD_F32 && dtype != DD_U8) return fail(DD_ERR_BAD_ARG, "dtype must be DD_F32 or DD_U8");
    if (ndm < 0 || nsamp < 0 || nbeams < 1) return fail(DD_ERR_BAD_ARG, "bad ndm / nsamp / nbeams");
    const int w = prm->median_window <= 1 ? 1 : prm->median_window;
    if (w != 1 && w != 3 && w != 5 && w != 7 && w != 9)
        return fail(DD_ERR_BAD_ARG, "median_window must be 0, 1, 3, 5, 7 or 9");
    if (prm->normalise && !prm->detrend)
        return fail(DD_ERR_BAD_ARG, "normalise needs detrend (the thesis normalises the detrended series)");
    if (prm->threshold_on && !prm->detrend)
        return fail(DD_ERR_BAD_ARG, "the n-sigma threshold needs detrend (sigma is the detrended series')");
    if (prm->threshold_on && (!cand || !count || capacity < 0))
        return fail(DD_ERR_BAD_ARG, "thresholding needs a candidate buffer and a counter");
    if (prm->threshold_on && !(prm->nsigma == prm->nsigma)) return fail(DD_ERR_BAD_ARG, "nsigma is NaN");
    if (ndm == 0 || nsamp == 0) return DD_OK;
    if (!D) return fail(DD_ERR_BAD_ARG, "D is null");
    if (nsamp > 2147483647LL) return fail(DD_ERR_BAD_ARG, "nsamp must fit int32 (candidate time index)");
    if (stride < nsamp || (Z && z_stride < nsamp)) return fail(DD_ERR_BAD_ARG, "stride is shorter than nsamp");
    if (nbeams > 1 && (beam_stride <= 0 || (Z && z_beam_stride <= 0)))
        return fail(DD_ERR_BAD_ARG, "beam strides must be positive when nbeams > 1");
    if (Z && (const void*)Z == D && w > 1)
        return fail(DD_ERR_BAD_ARG, "in-place output needs median_window <= 1 (neighbours read each other's samples)");
    const int64_t nrows = (int64_t)nbeams * ndm;
    // block steps per grid tile of the apply kernel: as many as still leave every SM a few waves of blocks
    int steps = kApplyJ;
    while (steps > 1 && nrows * ((nsamp + kTile * steps - 1) / (kTile * steps)) < 148 * 16) steps >>= 1;
    const int64_t ntiles = (nsamp + (int64_t)kTile * steps - 1) / ((int64_t)kTile * steps);
    if (nrows * ntiles > 2147483647LL) return fail(DD_ERR_UNSUPPORTED, "series x time tiles exceed one grid: split the call");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double* own_stats = nullptr;
    if (prm->detrend && !stats) {
        int rc = workspace_alloc((void**)&own_stats, (size_t)nrows * 3 * sizeof(double), cuda_stream);
        if (rc != DD_OK) return rc;
        stats = own_stats;
    }
    // candidates-only calls: the statistics pass leaves the largest median of every 128-sample chunk (4 bytes per
    // 512 of D), and the second pass reads D only in chunks that can hold a detection
    int32_t* cmax = nullptr;
    if (may_allocate && prm->detrend && prm->threshold_on && !Z && prm->nsigma >= 0.0f) {
        int rc = workspace_alloc((void**)&cmax, (size_t)nrows * (size_t)((nsamp + kChunk - 1) / kChunk) * 4, cuda_stream);
        if (rc != DD_OK) {
            if (own_stats) cudaFreeAsync(own_stats, st);
            return rc;
        }
    }
    ApplyParams ap{stride, nbeams > 1 ? beam_stride : 0, nsamp, ndm, (unsigned)ntiles, (unsigned)steps, prm->detrend, prm->normalise,
                   prm->threshold_on, (double)prm->nsigma, stats, cmax, Z, z_stride, nbeams > 1 ? z_beam_stride : 0,
                   cand, capacity, count};
    const int rc = dtype == DD_F32 ? launch_t<float>(w, D, nrows, ap, stats, st)
                                   : launch_t<int32_t>(w, D, nrows, ap, stats, st);
    if (own_stats) cudaFreeAsync(own_stats, st);
    if (cmax) cudaFreeAsync(cmax, st);
    return rc;
}

int postprocess(int dtype, const void* D, int64_t stride, int64_t beam_stride, int ndm, int64_t nsamp, int nbeams,
                const dd_post_params* prm, float* Z, int64_t z_stride, int64_t z_beam_stride, double* stats,
                dd_candidate* cand, int64_t capacity, unsigned long long* count, void* cuda_stream)
{
    return postprocess_impl(dtype, D, stride, beam_stride, ndm, nsamp, nbeams, prm, Z, z_stride, z_beam_stride, stats,
                            cand, capacity, count, cuda_stream, true);
}

// ---- the entry point that allocates nothing (dd_postprocess_static) --------------------------------
// The only scratch memory of the post-processing path is the table of per-series statistics (intercept,
// slope, sigma: 3 doubles per series) that the statistics kernel writes and the apply kernel reads.
// Here it lives in a file-scope device array (every GPU that loads the library holds these 384 KiB
// until exit), so the call reaches no cudaMalloc / cudaMallocAsync / cudaFree.  Every entry the apply kernel
// reads has been written by the statistics kernel of the SAME call (rows 0 .. nbeams*ndm-1), so nothing
// has to start at zero and nothing is cleared; the array keeps the last call's statistics.  All calls
// on one device share it: two calls that overlap on the GPU (different streams) race.
namespace {

constexpr int64_t kStaticMaxSeries = DD_POSTPROCESS_STATIC_MAX_SERIES;
static __device__ __align__(256) double g_static_stats[kStaticMaxSeries * 3];

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
double* g_static_addr[kStaticMaxDevices] = {};            // device address of g_static_stats, per device

// In host code `g_static_stats` is the host-side stand-in of the symbol, not a device address: the
// address is looked up once per device, with that device current.
int static_stats_address(double** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(DD_ERR_CUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(DD_ERR_UNSUPPORTED, "device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        double* ptr = nullptr;
        e = cudaGetSymbolAddress((void**)&ptr, g_static_stats);
        if (e != cudaSuccess || !ptr) {
            cudaGetLastError();
            return fail(DD_ERR_CUDA, std::string("cudaGetSymbolAddress(static statistics table): ") +
                                         cudaGetErrorString(e));
        }
        g_static_addr[dev] = ptr;
    }
    *out = g_static_addr[dev];
    return DD_OK;
}

}  // namespace

int postprocess_static(int dtype, const void* D, int64_t stride, int64_t beam_stride, int ndm, int64_t nsamp,
                       int nbeams, const dd_post_params* prm, float* Z, int64_t z_stride, int64_t z_beam_stride,
                       dd_candidate* cand, int64_t capacity, unsigned long long* count, void* cuda_stream)
{
    if (ndm < 0 || nbeams < 1) return fail(DD_ERR_BAD_ARG, "bad ndm / nbeams");
    if ((int64_t)nbeams * ndm > kStaticMaxSeries)
        return fail(DD_ERR_UNSUPPORTED,
                    "dd_postprocess_static: nbeams * ndm = " + std::to_string((int64_t)nbeams * ndm) +
                        " series exceed the static statistics table (DD_POSTPROCESS_STATIC_MAX_SERIES = " +
                        std::to_string(kStaticMaxSeries) + "); split the call or use dd_postprocess");
    double* stats = nullptr;
    const int rc = static_stats_address(&stats);
    if (rc != DD_OK) return rc;
    // with a statistics table passed in and the chunk-maximum workspace of candidates-only calls forgone (the second
    // pass then reads all of D, same candidates), nothing is allocated or freed
    return postprocess_impl(dtype, D, stride, beam_stride, ndm, nsamp, nbeams, prm, Z, z_stride, z_beam_stride, stats,
                            cand, capacity, count, cuda_stream, false);
}

}  // namespace dd
