// Coherent multi-beam beamformer, warp-level MMA kernel (the tcgen05 kernel of beamform_tc.cu takes arrays of up to
// 128 antennas; this one the wider ones) (ch. 5: eq 5.1, Alg. 2):
//     b(f, t, beam) = sum_a W[f][beam][a] * v[f][t][a],     P[beam][f][t] = |b|^2,
// v the 4-bit complex antenna voltages (one byte per antenna sample), W the phase
// weights held fixed over the buffer, P the detected beam power in the layout
// [beam][chan][time] that dd_execute takes as a multi-beam input -- the beams feed the dedisperser
// without leaving the device.
//
// "The beamforming process is essentially a matrix-vector multiplication ... per frequency channel"
// (PAPER.md:1639): a dense complex contraction with a tiny inner dimension (N_a antennas).  Written
// as a real product  [Re b; Im b] = [Wr -Wi; Wi Wr] [Re v; Im v]  it is a (2 N_b) x (2 N_a) x N_t GEMM per
// channel.  Roofline: per (f, t) the kernel reads N_a bytes and writes 4 N_b bytes for 8 N_a N_b flops
// -- 43 flop/B at 32 antennas x 16 beams, i.e. 275 Tflop/s to keep up with HBM: out of reach of the
// FP32 pipes (74 Tflop/s), so the products run on the tensor cores with FP32 accumulation.  The B
// operand is produced IN REGISTERS (nibbles -> fp16 pairs, exact) so the register-operand warp MMA
// (mma.sync m16n8k16) is the natural instruction: tcgen05 would need the unpacked voltages staged
// through shared memory (4x the bytes of the packed input) for a K of only 64.  The weights are split
// into two fp16 terms (hi + lo, |W - hi - lo| <= 2^-22 |W|), so the result has FP32 accuracy.
// Measured (32 antennas, 16 beams, 1024 channels x 2^16 samples): 2.6 ms = 2.4 TB/s = 37 % of the HBM copy
// bandwidth, 210 Tflop/s of fp16 MMAs issued (two per useful product).  What binds is the accumulate latency of
// the warp-level MMA at two to three warps per scheduler (154-164 registers): with the k-step loop outermost every
// MMA goes to a different accumulator (16 independent chains; 2.94 -> 2.63 ms); the tensor pipe is ~35 % busy, DRAM
// latency is not exposed (prefetching the next voltages into L2 changes nothing), more resident warps at 128
// registers spill.  The tcgen05 kernel (beamform_tc.cu) runs the same input in 1.36 ms.
// The thesis' kernel (Alg. 2) kept one FP32 accumulator per beam in registers and the weights in shared
// memory, and was bound by shared-memory requests.
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <algorithm>

#include "dd_internal.h"

namespace dd {

namespace {

constexpr int kWarps = 4;
constexpr int kNT = 8;                        // n-tiles (of 8 samples) per warp: 64 samples
constexpr int kWarpSamples = 8 * kNT;
constexpr int kKC = 4;                        // k-steps (of 8 antennas) whose weights sit in registers at a time

__device__ __forceinline__ void mma16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1)
{
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// one voltage byte (low nibble real, high nibble imaginary, 4-bit two's complement) -> (re, im) as fp16x2, exact:
// nibble n -> fp16 bits 0x6400 | (n ^ 8) = 1024 + (n + 8 mod 16), minus 1032
__device__ __forceinline__ uint32_t nibbles_to_half2(uint32_t byte)
{
    uint32_t t = (byte & 0x0fu) | ((byte & 0xf0u) << 12);
    t = (t ^ 0x00080008u) | 0x64006400u;
    const __half2 h = __hsub2(*reinterpret_cast<const __half2*>(&t), __floats2half2_rn(1032.0f, 1032.0f));
    return *reinterpret_cast<const uint32_t*>(&h);
}

// Weight preparation: W complex64 [nchans][nbeams][nants] -> A fragments of mma.m16n8k16 in the order the
// main kernel reads them: [chan][beam group of 8 MT][k-step][m-tile][lane][8 words: hi regs 0-3, lo regs 0-3].
// Row r < 8 of an m-tile is Re of beam 8 mt + r, row r + 8 its Im; column 2 a' + {0, 1} = (re, im) of antenna a'.
__global__ void __launch_bounds__(256)
dd_beamform_prepare_kernel(const float2* __restrict__ W, int nchans, int nbeams, int nants, int MT, int nbg, int KS,
                           uint32_t* __restrict__ A)
{
    const int64_t total = (int64_t)nchans * nbg * KS * MT * 32;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const int lane = (int)(i % 32);
        const int mt = (int)((i / 32) % MT);
        const int s = (int)((i / (32 * MT)) % KS);
        const int bg = (int)((i / ((int64_t)32 * MT * KS)) % nbg);
        const int f = (int)(i / ((int64_t)32 * MT * KS * nbg));
        const int g = lane >> 2, q = lane & 3;
        const int beam = (bg * MT + mt) * 8 + g;
        uint32_t hi[4], lo[4];
#pragma unroll
        for (int half = 0; half < 2; ++half) {                // antenna 8 s + q (regs 0, 1) and 8 s + q + 4 (regs 2, 3)
            const int a = 8 * s + q + 4 * half;
            float2 w = make_float2(0.0f, 0.0f);
            if (beam < nbeams && a < nants) w = W[((int64_t)f * nbeams + beam) * nants + a];
            // Re row: (Wr, -Wi); Im row: (Wi, Wr)
            const float v[2][2] = {{w.x, -w.y}, {w.y, w.x}};
#pragma unroll
            for (int row = 0; row < 2; ++row) {
                const __half h0 = __float2half_rn(v[row][0]), h1 = __float2half_rn(v[row][1]);
                const __half l0 = __float2half_rn(v[row][0] - __half2float(h0));
                const __half l1 = __float2half_rn(v[row][1] - __half2float(h1));
                const __half2 hh = __halves2half2(h0, h1), ll = __halves2half2(l0, l1);
                hi[2 * half + row] = *reinterpret_cast<const uint32_t*>(&hh);
                lo[2 * half + row] = *reinterpret_cast<const uint32_t*>(&ll);
            }
        }
        uint4* dst = reinterpret_cast<uint4*>(A + i * 8);
        dst[0] = make_uint4(hi[0], hi[1], hi[2], hi[3]);
        dst[1] = make_uint4(lo[0], lo[1], lo[2], lo[3]);
    }
}

// grid: (time tiles of kWarps * 64 samples, channel, beam group); a warp owns 64 samples.
template <int MT>
__global__ void __launch_bounds__(32 * kWarps)
dd_beamform_kernel(const uint8_t* __restrict__ V, const uint32_t* __restrict__ A, float* __restrict__ P, int nants,
                   int nchans, int64_t nsamp, int nbeams, int KS, int64_t out_stride, int64_t out_beam_stride)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane >> 2, q = lane & 3;
    const int f = blockIdx.y, bg = blockIdx.z, nbg = gridDim.z;
    const int64_t t0 = ((int64_t)blockIdx.x * kWarps + warp) * kWarpSamples;
    if (t0 >= nsamp) return;
    const uint32_t* vrow = reinterpret_cast<const uint32_t*>(V + (int64_t)f * nsamp * nants);   // nants % 4 == 0
    const int wps = nants / 4;                             // 32-bit words per sample
    float acc[MT][kNT][4];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
        for (int nt = 0; nt < kNT; ++nt)
#pragma unroll
            for (int e = 0; e < 4; ++e) acc[mt][nt][e] = 0.0f;

    for (int kc = 0; kc < KS; kc += kKC) {
        // this chunk's weights: registers, reused for all 64 samples
        uint32_t ah[kKC][MT][4], al[kKC][MT][4];
#pragma unroll
        for (int s = 0; s < kKC; ++s)
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                if (kc + s < KS) {
                    const uint4* src = reinterpret_cast<const uint4*>(
                        A + ((((int64_t)f * nbg + bg) * KS + kc + s) * MT + mt) * 256 + lane * 8);
                    const uint4 h = __ldg(src), l = __ldg(src + 1);
                    ah[s][mt][0] = h.x; ah[s][mt][1] = h.y; ah[s][mt][2] = h.z; ah[s][mt][3] = h.w;
                    al[s][mt][0] = l.x; al[s][mt][1] = l.y; al[s][mt][2] = l.z; al[s][mt][3] = l.w;
                } else {
#pragma unroll
                    for (int e = 0; e < 4; ++e) ah[s][mt][e] = al[s][mt][e] = 0u;
                }
            }
        // the chunk's 2 kKC words of every sample of the warp (the four lanes of a quad read the same words), all
        // loads first; then k-step outermost, so that consecutive MMAs go to different accumulators (16 independent
        // chains instead of two: the accumulate latency of the warp-level MMA is what two warps per scheduler expose)
        uint32_t w[kNT][2 * kKC];
#pragma unroll
        for (int nt = 0; nt < kNT; ++nt) {
            const int64_t t = min(t0 + 8 * nt + g, nsamp - 1);            // the tail repeats the last sample (never stored)
            const uint32_t* vs = vrow + t * wps + 2 * kc;
#pragma unroll
            for (int i = 0; i < 2 * kKC; ++i) w[nt][i] = (2 * kc + i < wps) ? __ldg(vs + i) : 0u;
        }
#pragma unroll
        for (int s = 0; s < kKC; ++s) {
#pragma unroll
            for (int nt = 0; nt < kNT; ++nt) {
                // B fragment of k-step s: antenna 8 s + q (word 2 s, byte q) and antenna 8 s + q + 4 (word 2 s + 1, byte q)
                const uint32_t b0 = nibbles_to_half2((w[nt][2 * s] >> (8 * q)) & 0xffu);
                const uint32_t b1 = nibbles_to_half2((w[nt][2 * s + 1] >> (8 * q)) & 0xffu);
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) mma16816(acc[mt][nt], ah[s][mt], b0, b1);
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) mma16816(acc[mt][nt], al[s][mt], b0, b1);
            }
        }
    }
    // detected power: rows g (Re) and g + 8 (Im) of beam 8 mt + g; columns 2 q, 2 q + 1 = samples
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
        const int beam = (bg * MT + mt) * 8 + g;
        if (beam >= nbeams) continue;
        float* prow = P + (int64_t)beam * out_beam_stride + (int64_t)f * out_stride;
#pragma unroll
        for (int nt = 0; nt < kNT; ++nt) {
            const int64_t t = t0 + 8 * nt + 2 * q;
            const float p0 = acc[mt][nt][0] * acc[mt][nt][0] + acc[mt][nt][2] * acc[mt][nt][2];
            const float p1 = acc[mt][nt][1] * acc[mt][nt][1] + acc[mt][nt][3] * acc[mt][nt][3];
            if (t + 1 < nsamp && ((((uintptr_t)(prow + t)) & 7) == 0)) {
                *reinterpret_cast<float2*>(prow + t) = make_float2(p0, p1);
            } else {
                if (t < nsamp) prow[t] = p0;
                if (t + 1 < nsamp) prow[t + 1] = p1;
            }
        }
    }
}

}  // namespace

int beamform_power_u4(const uint8_t* V, int nants, int nchans, int64_t nsamp, const float* W, int nbeams, float* P,
                      int64_t out_stride, int64_t out_beam_stride, void* cuda_stream)
{
    if (nants < 1 || nchans < 1 || nsamp < 0 || nbeams < 1) return fail(DD_ERR_BAD_ARG, "bad nants / nchans / nsamp / nbeams");
    if (nants % 4) return fail(DD_ERR_BAD_ARG, "nants must be a multiple of 4 (four antenna bytes per 32-bit word, PAPER.md:1645)");
    if (nsamp == 0) return DD_OK;
    if (!V || !W || !P) return fail(DD_ERR_BAD_ARG, "null pointer");
    if (((uintptr_t)V & 3) || ((uintptr_t)W & 7) || ((uintptr_t)P & 3)) return fail(DD_ERR_BAD_ARG, "misaligned pointer");
    if (out_stride < nsamp) return fail(DD_ERR_BAD_ARG, "out_stride is shorter than nsamp");
    if (nbeams > 1 && out_beam_stride < (int64_t)nchans * out_stride)
        return fail(DD_ERR_BAD_ARG, "out_beam_stride is shorter than a beam");
    // up to 128 antennas: the tcgen05 kernel (beamform_tc.cu); wider arrays: the warp-level MMA kernel below
    if (beamform_tc_ok(nants, nbeams))
        return beamform_tc_launch(V, nants, nchans, nsamp, W, nbeams, P, out_stride, out_beam_stride, cuda_stream);
    const int MT = nbeams > 8 ? 2 : 1;
    const int nbg = (nbeams + 8 * MT - 1) / (8 * MT);
    const int KS = (nants + 7) / 8;
    const int64_t ntile = (nsamp + kWarps * kWarpSamples - 1) / (kWarps * kWarpSamples);
    if (nchans > 65535 || nbg > 65535 || ntile > 2147483647LL)
        return fail(DD_ERR_UNSUPPORTED, "nchans / beam groups exceed one grid");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    uint32_t* A = nullptr;
    const size_t awords = (size_t)nchans * nbg * KS * MT * 32 * 8;
    int rc = workspace_alloc((void**)&A, awords * sizeof(uint32_t), cuda_stream);
    if (rc != DD_OK) return rc;
    dd_beamform_prepare_kernel<<<(unsigned)std::min<int64_t>(((int64_t)awords / 8 + 255) / 256, 4096), 256, 0, st>>>(
        reinterpret_cast<const float2*>(W), nchans, nbeams, nants, MT, nbg, KS, A);
    dim3 grid((unsigned)ntile, (unsigned)nchans, (unsigned)nbg);
    if (MT == 2)
        dd_beamform_kernel<2><<<grid, 32 * kWarps, 0, st>>>(V, A, P, nants, nchans, nsamp, nbeams, KS, out_stride,
                                                            out_beam_stride);
    else
        dd_beamform_kernel<1><<<grid, 32 * kWarps, 0, st>>>(V, A, P, nants, nchans, nsamp, nbeams, KS, out_stride,
                                                            out_beam_stride);
    cudaError_t e = cudaGetLastError();
    cudaFreeAsync(A, st);
    if (e != cudaSuccess) return fail(DD_ERR_CUDA, std::string("beamformer launch: ") + cudaGetErrorString(e));
    return DD_OK;
}

}  // namespace dd
