// uint8 front end: four byte-shifted copies of the input.
//
// A block of ps_u8.cu needs, for every channel, the window X[c][t0 + s(d0,c) ...) whose start has
// arbitrary byte alignment (PAPER.md:986 notes the misaligned loads), while TMA copies need
// 16-byte aligned sources (a byte-granular tensor-map coordinate faults on sm_100a: measured).
// This HBM-bound kernel therefore writes  W_r[row][i] = X[row][i + r],  r = 0..3,  into a padded
// workspace; a trial whose first operand sits at byte a then reads ALIGNED 32-bit words of copy
// (a & 3).  Layout [beam * nchans + channel][copy r][wcopy bytes]: the four copies of a channel
// are adjacent rows, so one 2-D tensor copy fetches the 16 rows of a four-channel group.
#include <cuda_runtime.h>

#include <algorithm>

#include "dd_internal.h"

namespace dd {

namespace {

constexpr int64_t kTailPad = 2048 + 16;   // a time tile may over-read its window by up to one tensor-copy box

// One thread per 16 output bytes of each copy; rows on grid.x (no 65535 limit on nbeams * nchans).
// With the row start rounded down to 16 bytes (sh = bytes cut off, 0..15), the 16 bytes of copy r at vector k
// are source bytes 16 k + sh + r ..: five consecutive words out of the three aligned vectors k, k+1, k+2, funnel-
// shifted by 8 ((sh + r) & 3) bits.  WO = sh >> 2 is a template argument (register arrays need static indices);
// copy r starts at word WO or WO + 1.  Only aligned vectors that hold at least one valid byte of the row are read
// (the rest count as 0), so no access leaves the pages of the caller's buffer.  Loads and stores are 16 bytes wide (the one-word-per-thread form took 0.22 ms of config 2's
// 4.50 ms step; this one 0.13 ms).
template <int WO>
__device__ __forceinline__ void shift_row(const uint4* __restrict__ srcv, uint8_t* __restrict__ dst, int64_t wcopy,
                                          int sh, int64_t nvec, int64_t lastv)
{
    const int sub = sh & 3;
    for (int64_t k = (int64_t)blockIdx.y * blockDim.x + threadIdx.x; k < nvec; k += (int64_t)gridDim.y * blockDim.x) {
        const uint4 z = make_uint4(0u, 0u, 0u, 0u);
        const uint4 q0 = k <= lastv ? __ldg(srcv + k) : z;
        const uint4 q1 = k + 1 <= lastv ? __ldg(srcv + k + 1) : z;
        const uint4 q2 = k + 2 <= lastv ? __ldg(srcv + k + 2) : z;
        const uint32_t w[12] = {q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, q1.z, q1.w, q2.x, q2.y, q2.z, q2.w};
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const bool up = sub + r >= 4;                              // copy r starts one word further
            const int bits = 8 * ((sub + r) & 3);
            uint32_t o[4];
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                const uint32_t lo = up ? w[WO + m + 1] : w[WO + m], hi = up ? w[WO + m + 2] : w[WO + m + 1];
                o[m] = __funnelshift_r(lo, hi, bits);
            }
            *reinterpret_cast<uint4*>(dst + r * wcopy + 16 * k) = make_uint4(o[0], o[1], o[2], o[3]);
        }
    }
}

__global__ void __launch_bounds__(256)
dd_shift_copies_u8(const uint8_t* __restrict__ X, uint8_t* __restrict__ W, int64_t wcopy, int64_t wpitch,
                   int nchans, int64_t rowlen, int64_t in_stride, int64_t in_beam_stride)
{
    const int64_t row = blockIdx.x;                                   // beam * nchans + channel
    const uint8_t* src = X + (row / nchans) * in_beam_stride + (row % nchans) * in_stride;
    const int sh = (int)((uintptr_t)src & 15);
    const uint4* srcv = reinterpret_cast<const uint4*>(src - sh);     // aligned vectors covering the row
    const int64_t nvec = (rowlen + 15) >> 4;                          // output vectors per copy (wcopy >= 16 nvec)
    const int64_t lastv = (sh + rowlen - 1) >> 4;                     // last aligned vector holding a valid byte
    uint8_t* dst = W + row * wpitch;
    switch (sh >> 2) {
        case 0: shift_row<0>(srcv, dst, wcopy, sh, nvec, lastv); break;
        case 1: shift_row<1>(srcv, dst, wcopy, sh, nvec, lastv); break;
        case 2: shift_row<2>(srcv, dst, wcopy, sh, nvec, lastv); break;
        default: shift_row<3>(srcv, dst, wcopy, sh, nvec, lastv); break;
    }
}

}  // namespace

// Allocates (stream-ordered) and fills the four byte-shifted copies.  Rows are padded so that the
// last time tile may over-read its window (the excess only feeds output samples >= nsamp_out,
// which are never stored).  The caller frees *W_out with cudaFreeAsync.
int make_shift_copies_u8(const dd_plan* p, const ExecArgs& a, uint8_t** W_out, int64_t* wcopy_out,
                         int64_t* wpitch_out)
{
    cudaStream_t st = (cudaStream_t)a.stream;
    const int64_t rowlen = a.nsamp_out + p->host.maxshift;            // valid samples per channel row
    const int64_t wcopy = (rowlen + kTailPad + 127) / 128 * 128;
    const int64_t wpitch = 4 * wcopy;
    const int64_t nrows = (int64_t)a.nbeams * p->nchans;
    uint8_t* W = nullptr;
    int rc = workspace_alloc((void**)&W, (size_t)(nrows * wpitch), a.stream);
    if (rc != DD_OK) return rc;
    const int64_t nvec = (rowlen + 15) / 16;
    dim3 grid((unsigned)nrows, (unsigned)std::min<int64_t>((nvec + 255) / 256, 64));
    dd_shift_copies_u8<<<grid, 256, 0, st>>>((const uint8_t*)a.X, W, wcopy, wpitch, p->nchans, rowlen,
                                             a.in_stride, a.in_beam_stride);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        cudaFreeAsync(W, st);
        return fail(DD_ERR_CUDA, std::string("uint8 front end launch: ") + cudaGetErrorString(e));
    }
    *W_out = W;
    *wcopy_out = wcopy;
    *wpitch_out = wpitch;
    return DD_OK;
}

}  // namespace dd
