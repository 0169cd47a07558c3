// Direct kernel for tiny plans: one thread per output element.
//
// A plan with a few dozen trials and channels (BASELINE.json configs[0]: 64 channels x 32 trials x
// 8192 samples = 1.7e7 adds = 0.45 us of work at the add roofline) is bound by launch latency and
// by how many SMs the grid reaches, not by any pipe: the tiled kernels give it 16 blocks on 148 SMs
// and a serial chain of per-group barriers.  Here the grid covers the output plane (DM, t)
// with one thread per element: the trial's row of the delay table goes to shared
// memory once, then every thread sums its nchans operands  X[c][t + s(d,c)]  (eq 2.1,
// PAPER.md:720-724) straight from global memory (the whole input of such a plan sits in L2; lanes
// run along time, so every load is a contiguous 128-byte / 32-byte segment), in the order
// c = 0, 1, 2, ... into one register.  Which plans take this kernel is decided from the plan
// alone (nchans * ndm <= kDirectMaxCells), never from the call's nsamp, so one-shot, batch and
// streaming calls of a plan add in the same order and stay bit-identical.
#include <cuda_runtime.h>

#include "dd_internal.h"

namespace dd {

namespace {

constexpr int kThreads = 256;

template <typename TIn> struct Acc;
template <> struct Acc<float>   { using type = float; };
template <> struct Acc<uint8_t> { using type = int32_t; };

template <typename TIn>
__global__ void __launch_bounds__(kThreads)
dd_direct_kernel(const TIn* __restrict__ X, typename Acc<TIn>::type* __restrict__ D,
                 const int32_t* __restrict__ shift, const int32_t* __restrict__ order, int nchans, int64_t nsamp,
                 int64_t in_stride, int64_t in_beam_stride, int64_t out_stride, int64_t out_beam_stride)
{
    using TAcc = typename Acc<TIn>::type;
    extern __shared__ int32_t sh[];                        // this trial's delays
    const int d = blockIdx.y;                              // sorted trial index
    for (int c = threadIdx.x; c < nchans; c += kThreads) sh[c] = shift[(int64_t)d * nchans + c];
    __syncthreads();
    const int64_t t = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (t >= nsamp) return;
    const TIn* x = X + (int64_t)blockIdx.z * in_beam_stride + t;
    TAcc acc = 0;
    int c = 0;
    for (; c + 8 <= nchans; c += 8) {
        TIn v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k] = __ldg(x + (int64_t)(c + k) * in_stride + sh[c + k]);
#pragma unroll
        for (int k = 0; k < 8; ++k) acc += (TAcc)v[k];
    }
    for (; c < nchans; ++c) acc += (TAcc)__ldg(x + (int64_t)c * in_stride + sh[c]);
    D[(int64_t)blockIdx.z * out_beam_stride + (int64_t)order[d] * out_stride + t] = acc;
}

template <typename TIn>
int launch_t(const ExecArgs& a)
{
    using TAcc = typename Acc<TIn>::type;
    const int64_t ntile_t = (a.nsamp_out + kThreads - 1) / kThreads;
    dim3 grid((unsigned)ntile_t, (unsigned)a.ndm, (unsigned)a.nbeams);
    dd_direct_kernel<TIn><<<grid, kThreads, (size_t)a.nchans * sizeof(int32_t), (cudaStream_t)a.stream>>>(
        (const TIn*)a.X, (TAcc*)a.D, a.d_shift, a.d_order, a.nchans, a.nsamp_out, a.in_stride, a.in_beam_stride,
        a.out_stride, a.out_beam_stride);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(DD_ERR_CUDA, std::string("direct launch: ") + cudaGetErrorString(e));
    return DD_OK;
}

}  // namespace

bool direct_args_ok(const ExecArgs& a)
{
    return a.ndm <= 65535 && a.nbeams <= 65535 && a.nchans <= 8192 &&
           (a.nsamp_out + kThreads - 1) / kThreads <= 2147483647LL;
}

int launch_direct(int dtype, const ExecArgs& a)
{
    if (dtype == DD_F32) return launch_t<float>(a);
    if (dtype == DD_U8) return launch_t<uint8_t>(a);
    return fail(DD_ERR_BAD_ARG, "bad dtype");
}

}  // namespace dd
