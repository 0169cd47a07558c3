// Generic "channel vector" kernel: works for ANY plan (unsorted / non-uniform DM lists, large
// per-trial shift steps, unaligned pointers and strides).  It is the correctness anchor and the
// fallback for plans the partial-sum kernels (ps_f32.cu, ps_u8.cu) do not take.
//
// Structure (the thesis' Alg. 1, modernised): the grid maps onto the output
// plane (DM, t); a block owns KB consecutive (sorted) trials x TB = 1024 output
// samples; for each channel the "channel vector" X[c][t0+s(d0,c) .. t0+TB+s(d_last,c)) (eq 2.14,
// PAPER.md:945) is staged in shared memory -- here CH channels at a time with cp.async, double
// buffered -- and every thread adds the shifted sample into KB x 4 register accumulators
// ("Accumulators are stored in registers").  Channels are added in the order
// c = 0,1,2,... for every output element, independent of the tile.
//
// Roofline: one shared-memory word per add -> at most 32 adds/clk/SM (25 % of the FP32 add
// pipe).  This is the thesis' design point ("roughly evenly split between single precision
// floating point, integer and shared memory access").
#include <cuda_runtime.h>

#include "dd_internal.h"

namespace dd {

namespace {

constexpr int kThreads = 256;
constexpr int kTPT = 4;                       // output samples per thread (stride kThreads)
constexpr int kTB = kThreads * kTPT;          // output samples per block
constexpr int kCH = 8;                        // channels staged per pipeline step

__device__ __forceinline__ void cp_async4(void* smem, const void* gmem)
{
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

template <typename TIn> struct Acc;
template <> struct Acc<float>   { using type = float; };
template <> struct Acc<uint8_t> { using type = int32_t; };

template <typename TIn, int KB>
__global__ void __launch_bounds__(kThreads)
dd_generic_kernel(const TIn* __restrict__ X, typename Acc<TIn>::type* __restrict__ D,
                  const int32_t* __restrict__ shift, const int32_t* __restrict__ order,
                  int nchans, int ndm, int64_t nsamp, int64_t in_stride, int64_t in_beam_stride,
                  int64_t out_stride, int64_t out_beam_stride, int rowwords)
{
    using TAcc = typename Acc<TIn>::type;
    constexpr int EPW = 4 / (int)sizeof(TIn);            // elements per 32-bit staged word
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t* rows = smem;                                // [2][kCH][rowwords]
    int* offs = (int*)(smem + 2 * kCH * rowwords);        // [2][kCH][KB]

    const int tid = threadIdx.x;
    const int d0 = blockIdx.x * KB;                       // DM tiles fastest: the staged windows of
    const int64_t t0 = (int64_t)blockIdx.y * kTB;         // neighbouring blocks overlap in L2
    const int dl = min(d0 + KB, ndm) - 1;
    const TIn* Xb = X + (int64_t)blockIdx.z * in_beam_stride;
    const int32_t* tab0 = shift + (int64_t)d0 * nchans;
    const int32_t* tabl = shift + (int64_t)dl * nchans;

    TAcc acc[KB][kTPT];
#pragma unroll
    for (int j = 0; j < KB; ++j)
#pragma unroll
        for (int i = 0; i < kTPT; ++i) acc[j][i] = 0;

    const int ngroups = (nchans + kCH - 1) / kCH;

    auto stage = [&](int g, int buf) {
        const int c0 = g * kCH;
        if (tid < kCH * KB) {
            const int ch = tid / KB, j = tid % KB;
            const int c = c0 + ch;
            if (c < nchans) {
                const int d = min(d0 + j, ndm - 1);
                const int s0 = tab0[c];
                int o = shift[(int64_t)d * nchans + c] - s0;
                if (EPW > 1) {
                    const TIn* p = Xb + (int64_t)c * in_stride + t0 + s0;
                    o += (int)((uintptr_t)p & 3);
                }
                offs[(buf * kCH + ch) * KB + j] = o;
            }
        }
#pragma unroll 1
        for (int ch = 0; ch < kCH; ++ch) {
            const int c = c0 + ch;
            if (c >= nchans) break;
            const int s0 = tab0[c], sl = tabl[c];
            const int64_t e0 = t0 + s0;                               // first element needed
            int64_t need = min((int64_t)kTB + (sl - s0), nsamp + sl - e0);   // elements needed
            const TIn* p = Xb + (int64_t)c * in_stride + e0;
            const int resid = (EPW > 1) ? (int)((uintptr_t)p & 3) : 0;
            const uint32_t* wp = (const uint32_t*)((const char*)p - resid);
            const int nw = (int)((resid + need + EPW - 1) / EPW);
            uint32_t* row = rows + (size_t)(buf * kCH + ch) * rowwords;
            for (int w = tid; w < nw; w += kThreads) cp_async4(row + w, wp + w);
        }
        cp_async_commit();
    };

    stage(0, 0);
    for (int g = 0; g < ngroups; ++g) {
        const int buf = g & 1;
        if (g + 1 < ngroups) {
            stage(g + 1, buf ^ 1);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        __syncthreads();
        const int nch = min(kCH, nchans - g * kCH);
#pragma unroll 1
        for (int ch = 0; ch < nch; ++ch) {
            const TIn* row = (const TIn*)(rows + (size_t)(buf * kCH + ch) * rowwords) + tid;
            const int* o = offs + (buf * kCH + ch) * KB;
#pragma unroll
            for (int j = 0; j < KB; ++j) {
                const TIn* r = row + o[j];
#pragma unroll
                for (int i = 0; i < kTPT; ++i) acc[j][i] += (TAcc)r[i * kThreads];
            }
        }
        __syncthreads();
    }

    TAcc* Db = D + (int64_t)blockIdx.z * out_beam_stride;
#pragma unroll
    for (int j = 0; j < KB; ++j) {
        const int d = d0 + j;
        if (d >= ndm) break;
        TAcc* drow = Db + (int64_t)order[d] * out_stride;
#pragma unroll
        for (int i = 0; i < kTPT; ++i) {
            const int64_t t = t0 + tid + i * kThreads;
            if (t < nsamp) drow[t] = acc[j][i];
        }
    }
}

template <typename TIn, int KB>
int launch_one(const ExecArgs& a, int max_spread)
{
    using TAcc = typename Acc<TIn>::type;
    constexpr int EPW = 4 / (int)sizeof(TIn);
    const int rowwords = (kTB + max_spread + EPW - 1) / EPW + (EPW > 1 ? 1 : 0);
    const size_t smem = (size_t)2 * kCH * rowwords * 4 + (size_t)2 * kCH * KB * 4;
    auto kern = dd_generic_kernel<TIn, KB>;
    int rc = ensure_dyn_smem((const void*)kern, smem);
    if (rc != DD_OK) return rc;
    cudaError_t e;
    const int64_t ntile_t = (a.nsamp_out + kTB - 1) / kTB;
    if (ntile_t > 65535 || a.nbeams > 65535)
        return fail(DD_ERR_UNSUPPORTED, "nsamp_out / nbeams too large for one launch");
    dim3 grid((unsigned)((a.ndm + KB - 1) / KB), (unsigned)ntile_t, (unsigned)a.nbeams);
    kern<<<grid, kThreads, smem, (cudaStream_t)a.stream>>>(
        (const TIn*)a.X, (TAcc*)a.D, a.d_shift, a.d_order, a.nchans, a.ndm, a.nsamp_out,
        a.in_stride, a.in_beam_stride, a.out_stride, a.out_beam_stride, rowwords);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(DD_ERR_CUDA, std::string("generic launch: ") + cudaGetErrorString(e));
    return DD_OK;
}

template <typename TIn>
int launch_kb(int kb, int max_spread, const ExecArgs& a)
{
    switch (kb) {
        case 16: return launch_one<TIn, 16>(a, max_spread);
        case 8:  return launch_one<TIn, 8>(a, max_spread);
        case 4:  return launch_one<TIn, 4>(a, max_spread);
        case 2:  return launch_one<TIn, 2>(a, max_spread);
        case 1:  return launch_one<TIn, 1>(a, max_spread);
    }
    return fail(DD_ERR_BAD_ARG, "generic kernel: bad KB");
}

}  // namespace

int launch_generic(int dtype, int kb, int max_spread, const ExecArgs& a)
{
    if (dtype == DD_F32) return launch_kb<float>(kb, max_spread, a);
    if (dtype == DD_U8) return launch_kb<uint8_t>(kb, max_spread, a);
    return fail(DD_ERR_BAD_ARG, "bad dtype");
}

}  // namespace dd
