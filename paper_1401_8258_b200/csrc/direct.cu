// Direct kernel for tiny plans: operands straight from global memory / L2.
//
// A plan with a few dozen trials and channels (BASELINE.json configs[0]: 64 channels x 32 trials x
// 8192 samples = 1.7e7 adds = 0.45 us of work at the add roofline) is bound by launch latency and
// by memory latency, not by any pipe: the tiled kernels give it 16 blocks on 148 SMs and a
// serial chain of per-group barriers.  Here the grid covers the output plane (DM, t)
// (PAPER.md:956): a block owns 128 output samples of 4 adjacent trials and has 4 x 128 threads;
// the trials' rows of the delay table go to shared memory once; thread (x, q) sums, for each of
// the 4 trials, the operands  X[c][t + s(d,c)]  (eq 2.1) of the q-th quarter of
// the channels, in ascending channel order, straight from global memory (the whole input of
// such a plan sits in L2, the overlapping windows of adjacent trials are served by L1; lanes run
// along time, so every load is a contiguous segment); the four partial sums of an output meet in
// shared memory and are added as ((p0 + p1) + p2) + p3.  Splitting the channels keeps 55 warps
// per SM in flight -- the kernel is latency-bound (ncu: long-scoreboard stalls, no pipe above
// 15 %).  Which plans take this kernel is decided from the plan alone (nchans * ndm <=
// kDirectMaxCells), never from the call's nsamp, so one-shot, batch and streaming calls of a
// plan add in the same order and stay bit-identical.
#include <cuda_runtime.h>

#include "dd_internal.h"

namespace dd {

namespace {

constexpr int kTX = 128;                      // output samples per block
constexpr int kQ = 4;                         // channel quarters: threadIdx.y; partial sums meet in shared memory
constexpr int kKD = 4;                        // adjacent (sorted) trials per block: their windows overlap in L1
constexpr int kCU = 8;                        // channels of loads in flight per thread
constexpr int kMaxChans = 4096;               // delays of all channels of the block's trials sit in shared memory

template <typename TIn> struct Acc;
template <> struct Acc<float>   { using type = float; };
template <> struct Acc<uint8_t> { using type = int32_t; };

template <typename TIn>
__global__ void __launch_bounds__(kTX * kQ)
dd_direct_kernel(const TIn* __restrict__ X, typename Acc<TIn>::type* __restrict__ D,
                 const int32_t* __restrict__ shift, const int32_t* __restrict__ order, int nchans, int ndm,
                 int64_t nsamp, int64_t in_stride, int64_t in_beam_stride, int64_t out_stride,
                 int64_t out_beam_stride)
{
    using TAcc = typename Acc<TIn>::type;
    extern __shared__ __align__(16) int32_t dsm[];
    TAcc* part = reinterpret_cast<TAcc*>(dsm);             // [kQ][kKD][kTX] partial sums
    int32_t* sh = dsm + kQ * kKD * kTX;                    // [nchans][kKD] delays of this block's trials
    const int tx = threadIdx.x, q = threadIdx.y;
    const int d0 = blockIdx.y * kKD;                       // sorted trial index of the first one
    for (int i = q * kTX + tx; i < nchans * kKD; i += kTX * kQ) {
        const int c = i / kKD, j = i % kKD;
        sh[i] = shift[(int64_t)min(d0 + j, ndm - 1) * nchans + c];
    }
    __syncthreads();
    const int64_t t = (int64_t)blockIdx.x * kTX + tx;
    const TIn* x = X + (int64_t)blockIdx.z * in_beam_stride + min(t, nsamp - 1);
    // quarter q adds channels [c_lo, c_hi) in ascending order
    const int cq = (nchans + kQ - 1) / kQ;
    const int c_lo = min(nchans, q * cq), c_hi = min(nchans, c_lo + cq);
    TAcc acc[kKD];
#pragma unroll
    for (int j = 0; j < kKD; ++j) acc[j] = 0;
    int c = c_lo;
    for (; c + kCU <= c_hi; c += kCU) {
        // one trial at a time: the first trial's loads bring the lines into L1, the other trials'
        // windows (a few samples further) then hit there
#pragma unroll
        for (int j = 0; j < kKD; ++j) {
            TIn v[kCU];
#pragma unroll
            for (int k = 0; k < kCU; ++k) v[k] = __ldg(x + (int64_t)(c + k) * in_stride + sh[(c + k) * kKD + j]);
#pragma unroll
            for (int k = 0; k < kCU; ++k) acc[j] += (TAcc)v[k];
        }
    }
    for (; c < c_hi; ++c) {
#pragma unroll
        for (int j = 0; j < kKD; ++j) acc[j] += (TAcc)__ldg(x + (int64_t)c * in_stride + sh[c * kKD + j]);
    }
#pragma unroll
    for (int j = 0; j < kKD; ++j) part[(q * kKD + j) * kTX + tx] = acc[j];
    __syncthreads();
    // quarter q finishes trial q of the block: ((p0 + p1) + p2) + p3, the same order for every element
    if (t < nsamp && d0 + q < ndm) {
        TAcc v = part[(0 * kKD + q) * kTX + tx];
#pragma unroll
        for (int qq = 1; qq < kQ; ++qq) v += part[(qq * kKD + q) * kTX + tx];
        D[(int64_t)blockIdx.z * out_beam_stride + (int64_t)order[d0 + q] * out_stride + t] = v;
    }
}

template <typename TIn>
int launch_t(const ExecArgs& a)
{
    using TAcc = typename Acc<TIn>::type;
    static_assert(kQ == kKD, "quarter q stores trial q");
    const int64_t ntile_t = (a.nsamp_out + kTX - 1) / kTX;
    dim3 grid((unsigned)ntile_t, (unsigned)((a.ndm + kKD - 1) / kKD), (unsigned)a.nbeams);
    const size_t smem = (size_t)(kQ * kKD * kTX + a.nchans * kKD) * 4;
    int rc = ensure_dyn_smem((const void*)dd_direct_kernel<TIn>, smem);
    if (rc != DD_OK) return rc;
    dd_direct_kernel<TIn><<<grid, dim3(kTX, kQ), smem, (cudaStream_t)a.stream>>>(
        (const TIn*)a.X, (TAcc*)a.D, a.d_shift, a.d_order, a.nchans, a.ndm, a.nsamp_out, a.in_stride,
        a.in_beam_stride, a.out_stride, a.out_beam_stride);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(DD_ERR_CUDA, std::string("direct launch: ") + cudaGetErrorString(e));
    return DD_OK;
}

}  // namespace

bool direct_args_ok(const ExecArgs& a)
{
    return (a.ndm + kKD - 1) / kKD <= 65535 && a.nbeams <= 65535 && a.nchans <= kMaxChans &&
           (a.nsamp_out + kTX - 1) / kTX <= 2147483647LL;
}

int launch_direct(int dtype, const ExecArgs& a)
{
    if (dtype == DD_F32) return launch_t<float>(a);
    if (dtype == DD_U8) return launch_t<uint8_t>(a);
    return fail(DD_ERR_BAD_ARG, "bad dtype");
}

}  // namespace dd
