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

// One thread per output word; rows on grid.x (no 65535 limit on nbeams * nchans).
__global__ void __launch_bounds__(256)
dd_shift_copies_u8(const uint8_t* __restrict__ X, uint8_t* __restrict__ W, int64_t wcopy, int64_t wpitch,
                   int nchans, int64_t rowlen, int64_t in_stride, int64_t in_beam_stride)
{
    const int64_t row = blockIdx.x;                                   // beam * nchans + channel
    const uint8_t* src = X + (row / nchans) * in_beam_stride + (row % nchans) * in_stride;
    const int sh = (int)((uintptr_t)src & 3);
    const uint32_t* srcw = reinterpret_cast<const uint32_t*>(src - sh);   // aligned words covering the row
    const int64_t nwords = (rowlen + 3) >> 2;
    const int64_t lastw = (sh + rowlen - 1) >> 2;                     // last aligned word holding a valid byte
    for (int64_t i = (int64_t)blockIdx.y * blockDim.x + threadIdx.x; i < nwords;
         i += (int64_t)gridDim.y * blockDim.x) {
        const uint32_t w0 = __ldg(srcw + i);
        const uint32_t w1 = i + 1 <= lastw ? __ldg(srcw + i + 1) : 0u;
        const uint32_t w2 = i + 2 <= lastw ? __ldg(srcw + i + 2) : 0u;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int b = sh + r;                                     // 0..6 bytes into (w0,w1,w2)
            const uint32_t lo = b < 4 ? w0 : w1, hi = b < 4 ? w1 : w2;
            const uint32_t v = __funnelshift_r(lo, hi, 8 * (b & 3));
            reinterpret_cast<uint32_t*>(W + r * wcopy + row * wpitch)[i] = v;
        }
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
    const int64_t nwords = (rowlen + 3) / 4;
    dim3 grid((unsigned)nrows, (unsigned)std::min<int64_t>((nwords + 255) / 256, 64));
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
