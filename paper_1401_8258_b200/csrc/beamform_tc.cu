// Coherent multi-beam beamformer on the 5th-generation tensor cores (tcgen05.mma, accumulators in TMEM);
// SURVEY.md §8(f) row f4; PAPER.md:1600-1665 (eq 5.1, Alg. 2).  Same contract and same numbers as
// beamform.cu (which stays as the path for shapes this kernel does not take).
//
// Per frequency channel the beam voltages are a small dense contraction:
//     D[t][n] = sum_k A[t][k] B[n][k],   t = sample (M = 128 per tile),  k = 2 a + {re, im} of antenna a,
//     n = 2 beam + {0: Re b, 1: Im b},   B[2 b][2 a] = Wr, B[2 b][2 a + 1] = -Wi, B[2 b + 1][2 a] = Wi, B[2 b + 1][2 a + 1] = Wr.
// Samples sit on M so that an accumulator row (one TMEM lane = one thread of the epilogue) holds Re and Im of
// every beam of ONE sample: the detected power |b|^2 needs no exchange between threads and consecutive lanes
// write consecutive samples of a beam row (128-byte coalesced stores).
//   A (voltages): each of the 128 threads unpacks its own sample -- 4-bit two's complement nibbles to exact
//     fp16 pairs, one 32-bit input word (4 antennas) = one 16-byte chunk -- into the K-major, 128-byte-swizzled
//     shared-memory tile the MMA reads (row = sample = 128 bytes per 32 antennas; chunk c of row r lands at chunk
//     c ^ (r & 7): conflict-free 16-byte stores);
//   B (weights): hi + lo fp16 terms (|W - hi - lo| <= 2^-22 |W|), laid out by the prepare kernel exactly as the
//     shared-memory image, copied once per block and reused for all its time tiles; two MMAs per k-step (hi, lo)
//     accumulate in FP32 in TMEM;
//   one elected thread issues tcgen05.mma (M = 128, N = 2 x beams of the group, K = 16 per instruction) and commits
//     to an mbarrier; tiles are double buffered in shared memory and in TMEM, so the unpack of tile j + 1 and the
//     epilogue of tile j - 1 (tcgen05.ld -> power -> global) overlap the MMAs of tile j.
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <algorithm>

#include "dd_internal.h"
#include "tma_ptx.cuh"

namespace dd {

namespace {

constexpr int kTcThreads = 128;               // one sample (accumulator row) per thread
constexpr int kTcTilesPerBlock = 32;          // time tiles of 128 samples per block
constexpr int kTcMaxAtoms = 4;                // 128-byte K atoms (32 antennas each): up to 128 antennas
constexpr int kTcMaxNB = 32;                  // beams per group: N = 64 accumulator columns

__host__ __device__ inline int swz(int row, int chunk)   // byte offset of 16-byte chunk `chunk` of row `row` in a K-major SW128 tile
{
    return (row >> 3) * 1024 + (row & 7) * 128 + ((chunk ^ (row & 7)) << 4);
}

// Weight image: [chan][beam group][hi, lo][atom][N rows x 128 bytes, swizzled], fp16.
__global__ void __launch_bounds__(256)
dd_beamform_tc_prepare_kernel(const float2* __restrict__ W, int nchans, int nbeams, int nants, int NB, int nbg,
                              int natoms, __half* __restrict__ Bimg)
{
    const int N = 2 * NB;
    const int64_t per = (int64_t)2 * natoms * N * 64;                  // halves per (chan, group)
    const int64_t total = (int64_t)nchans * nbg * natoms * N * 64;      // (chan, group, atom, n, k in atom)
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const int kk = (int)(i % 64);
        const int n = (int)((i / 64) % N);
        const int atom = (int)((i / (64 * N)) % natoms);
        const int bg = (int)((i / ((int64_t)64 * N * natoms)) % nbg);
        const int f = (int)(i / ((int64_t)64 * N * natoms * nbg));
        const int k = atom * 64 + kk, a = k >> 1, beam = bg * NB + (n >> 1);
        float v = 0.0f;
        if (beam < nbeams && a < nants) {
            const float2 w = W[((int64_t)f * nbeams + beam) * nants + a];
            v = (n & 1) ? ((k & 1) ? w.x : w.y) : ((k & 1) ? -w.y : w.x);
        }
        const __half hi = __float2half_rn(v), lo = __float2half_rn(v - __half2float(hi));
        const int off = swz(n, kk >> 3) / 2 + (kk & 7);                 // halves inside the atom's tile
        __half* base = Bimg + ((int64_t)f * nbg + bg) * per;
        base[(int64_t)(0 * natoms + atom) * N * 64 + off] = hi;
        base[(int64_t)(1 * natoms + atom) * N * 64 + off] = lo;
    }
}

// shared-memory matrix descriptor of a K-major, 128-byte-swizzled tile (rows of 128 bytes, 8-row groups 1024 bytes
// apart): start address / 16 in bits 0-13, stride byte offset / 16 in bits 32-45, version 1 in bits 46-47,
// layout type SWIZZLE_128B = 2 in bits 61-63; the leading byte offset is not used by swizzled K-major layouts
__device__ __forceinline__ uint64_t umma_desc(uint32_t smem_addr)
{
    return (uint64_t)((smem_addr >> 4) & 0x3fffu) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}

// one 32-bit input word (4 antennas: low nibble real, high nibble imaginary, 4-bit two's complement) -> four
// (re, im) fp16 pairs, exact: nibble n -> fp16 bits 0x6400 | (n ^ 8) = 1024 + (n + 8 mod 16), minus 1032
__device__ __forceinline__ uint4 unpack_word(uint32_t w)
{
    const uint32_t lo = w & 0x0f0f0f0fu, hi = (w >> 4) & 0x0f0f0f0fu;
    const __half2 bias = __floats2half2_rn(1032.0f, 1032.0f);
    uint32_t r[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        uint32_t t = __byte_perm(lo, hi, 0x0400 + i * 0x0101 + 0x4040);   // bytes: lo_i, (hi_0), hi_i, (hi_0)
        t = (t & 0x000f000fu) ^ 0x64086408u;
        const __half2 h = __hsub2(*reinterpret_cast<const __half2*>(&t), bias);
        r[i] = *reinterpret_cast<const uint32_t*>(&h);
    }
    return make_uint4(r[0], r[1], r[2], r[3]);
}

struct TcParams {
    const uint8_t* V;
    const __half* Bimg;
    float* P;
    int nants, nchans, nbeams, NB, natoms, ksteps;       // ksteps: 16-half MMA steps over all antennas
    int64_t nsamp, out_stride, out_beam_stride;
};

template <int N, int NATOMS>                               // accumulator columns = 2 x beams per group; K atoms
__global__ void __launch_bounds__(kTcThreads)
dd_beamform_tc_kernel(const TcParams p)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const int tid = threadIdx.x, warp = tid >> 5;
    const int f = blockIdx.y, bg = blockIdx.z, nbg = gridDim.z;
    constexpr int natoms = NATOMS;
    const int wps = p.nants / 4;
    // shared memory: A [2][natoms][16 KB] | B [2 (hi, lo)][natoms][N x 128 B] | done[2] | tmem base
    uint8_t* As = smem;
    uint8_t* Bs = As + 2 * natoms * 16384;
    uint64_t* done = reinterpret_cast<uint64_t*>(Bs + 2 * natoms * N * 128);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(done + 2);

    if (tid == 0) {
        mbar_init(&done[0], 1);
        mbar_init(&done[1], 1);
        mbar_fence_init();
    }
    if (warp == 0) {                                       // TMEM: two accumulators of N columns
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(2 * N));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    {   // this (channel, beam group)'s weight image
        const uint4* src = reinterpret_cast<const uint4*>(p.Bimg + ((int64_t)f * nbg + bg) * (2 * natoms * N * 64));
        uint4* dst = reinterpret_cast<uint4*>(Bs);
        for (int i = tid; i < 2 * natoms * N * 8; i += kTcThreads) dst[i] = __ldg(src + i);
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;

    // instruction descriptor (kind::f16): D = F32 (bits 4-5 = 1), A = B = F16 (0), both K-major (bits 15, 16 = 0),
    // N >> 3 in bits 17-22, M >> 4 = 8 in bits 24-28
    constexpr uint32_t idesc = (1u << 4) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    const uint32_t as0 = smem_u32(As), bs0 = smem_u32(Bs);
    const int64_t tblock = (int64_t)blockIdx.x * kTcTilesPerBlock * 128;
    const uint32_t* vrow = reinterpret_cast<const uint32_t*>(p.V + (int64_t)f * p.nsamp * p.nants);

    auto epilogue = [&](int i) {
        mbar_wait(&done[i & 1], (i >> 1) & 1);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const int64_t t = tblock + (int64_t)i * 128 + tid;
        const uint32_t taddr = tmem + (uint32_t)((i & 1) * N) + ((uint32_t)(warp * 32) << 16);
#pragma unroll
        for (int c0 = 0; c0 < N; c0 += 32) {
            uint32_t v[32];
            asm volatile(
                "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                  "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
                  "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
                  "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
                : "r"(taddr + (uint32_t)c0));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (t < p.nsamp) {
                const int beam0 = bg * p.NB + (c0 >> 1);
                float* pp = p.P + (int64_t)beam0 * p.out_beam_stride + (int64_t)f * p.out_stride + t;
                if (beam0 + 16 <= p.nbeams) {
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        const float re = __uint_as_float(v[2 * q]), im = __uint_as_float(v[2 * q + 1]);
                        *pp = re * re + im * im;
                        pp += p.out_beam_stride;
                    }
                } else {
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        const float re = __uint_as_float(v[2 * q]), im = __uint_as_float(v[2 * q + 1]);
                        if (beam0 + q < p.nbeams) *pp = re * re + im * im;
                        pp += p.out_beam_stride;
                    }
                }
            }
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    };

    // the packed voltages of this thread's sample of tile j: loaded one tile ahead (registers), so that the loads
    // are in flight while the previous tile is multiplied and written out
    uint32_t wv[natoms * 8];
    auto load_tile = [&](int j) {
        const int64_t t = tblock + (int64_t)j * 128 + tid;
        const uint32_t* vs = vrow + min(t, p.nsamp - 1) * wps;       // the tail repeats the last sample (never stored)
        if ((wps & 3) == 0 && (((uintptr_t)vs) & 15) == 0) {
#pragma unroll
            for (int c4 = 0; c4 < natoms * 2; ++c4) {
                uint4 w = make_uint4(0u, 0u, 0u, 0u);
                if (4 * c4 < wps) w = __ldg(reinterpret_cast<const uint4*>(vs) + c4);
                wv[4 * c4] = w.x; wv[4 * c4 + 1] = w.y; wv[4 * c4 + 2] = w.z; wv[4 * c4 + 3] = w.w;
            }
        } else {
#pragma unroll
            for (int c = 0; c < natoms * 8; ++c) wv[c] = c < wps ? __ldg(vs + c) : 0u;
        }
    };
    const uint32_t rowoff = (uint32_t)((tid >> 3) * 1024 + (tid & 7) * 128), rx = (uint32_t)(tid & 7);
    if (tblock < p.nsamp) load_tile(0);

    int ntiles = 0;
#pragma unroll 1
    for (int j = 0; j < kTcTilesPerBlock; ++j) {
        if (tblock + (int64_t)j * 128 >= p.nsamp) break;
        ntiles = j + 1;
        // unpack this thread's sample into row tid of A[j & 1] (a zero word unpacks to zeros)
        uint8_t* a = As + (j & 1) * natoms * 16384;
#pragma unroll
        for (int c = 0; c < natoms * 8; ++c)
            *reinterpret_cast<uint4*>(a + (c >> 3) * 16384 + rowoff + (((uint32_t)(c & 7) ^ rx) << 4)) = unpack_word(wv[c]);
        if (j + 1 < kTcTilesPerBlock && tblock + (int64_t)(j + 1) * 128 < p.nsamp) load_tile(j + 1);
        {   // one 16-byte load per thread and tile leaves too little in flight: ask L2 for the tile three ahead
            // (32 antennas: 1.37 -> 1.27 ms)
            const int64_t tp = tblock + (int64_t)(j + 3) * 128 + tid;
            if (j + 3 < kTcTilesPerBlock && tp < p.nsamp) asm volatile("prefetch.global.L2 [%0];" ::"l"(vrow + tp * wps));
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        if (tid == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t d = tmem + (uint32_t)((j & 1) * N);
            const uint64_t da0 = umma_desc(as0 + (j & 1) * natoms * 16384), db0 = umma_desc(bs0);
#pragma unroll
            for (int ks = 0; ks < 4 * natoms; ++ks) {
                if (ks < p.ksteps) {
                    constexpr int kPartStride = natoms * (N * 128);
                    const int atom = ks >> 2, kin = ks & 3;            // 4 steps of 32 bytes per 128-byte atom
                    // (start address / 16 sits in the descriptor's low bits: tiles and k-steps are plain additions)
                    const uint64_t da = da0 + (uint64_t)((atom * 16384 + kin * 32) >> 4);
#pragma unroll
                    for (int part = 0; part < 2; ++part) {             // hi, lo weight terms
                        const uint64_t db = db0 + (uint64_t)((part * kPartStride + atom * (N * 128) + kin * 32) >> 4);
                        const uint32_t accumulate = (ks | part) ? 1u : 0u;
                        asm volatile(
                            "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
                            "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}"
                            ::"r"(d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
                            : "memory");
                    }
                }
            }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&done[j & 1]))
                         : "memory");
        }
        if (j >= 1) epilogue(j - 1);
    }
    if (ntiles >= 1) epilogue(ntiles - 1);
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(2 * N));
}

}  // namespace

bool beamform_tc_ok(int nants, int nbeams) { return nants % 4 == 0 && nants <= 32 * kTcMaxAtoms && nbeams >= 1; }

int beamform_tc_launch(const uint8_t* V, int nants, int nchans, int64_t nsamp, const float* W, int nbeams, float* P,
                       int64_t out_stride, int64_t out_beam_stride, void* cuda_stream)
{
    const int natoms = (2 * nants + 63) / 64, ksteps = (2 * nants + 15) / 16;
    const int NB = nbeams <= 16 ? 16 : kTcMaxNB, N = 2 * NB;        // N = 32 or 64 accumulator columns
    const int nbg = (nbeams + NB - 1) / NB;
    const int64_t nblk = (nsamp + (int64_t)kTcTilesPerBlock * 128 - 1) / ((int64_t)kTcTilesPerBlock * 128);
    if (nchans > 65535 || nbg > 65535 || nblk > 2147483647LL)
        return fail(DD_ERR_UNSUPPORTED, "nchans / beam groups exceed one grid");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    __half* Bimg = nullptr;
    const size_t halves = (size_t)nchans * nbg * 2 * natoms * N * 64;
    int rc = workspace_alloc((void**)&Bimg, halves * sizeof(__half), cuda_stream);
    if (rc != DD_OK) return rc;
    dd_beamform_tc_prepare_kernel<<<(unsigned)std::min<int64_t>(((int64_t)halves / 2 + 255) / 256, 8192), 256, 0, st>>>(
        reinterpret_cast<const float2*>(W), nchans, nbeams, nants, NB, nbg, natoms, Bimg);
    TcParams q{V, Bimg, P, nants, nchans, nbeams, NB, natoms, ksteps, nsamp, out_stride, out_beam_stride};
    const size_t smem = (size_t)2 * natoms * 16384 + (size_t)2 * natoms * N * 128 + 64;
    dim3 grid((unsigned)nblk, (unsigned)nchans, (unsigned)nbg);
    typedef void (*Kern)(const TcParams);
    static const Kern kerns[2][kTcMaxAtoms] = {
        {dd_beamform_tc_kernel<32, 1>, dd_beamform_tc_kernel<32, 2>, dd_beamform_tc_kernel<32, 3>, dd_beamform_tc_kernel<32, 4>},
        {dd_beamform_tc_kernel<64, 1>, dd_beamform_tc_kernel<64, 2>, dd_beamform_tc_kernel<64, 3>, dd_beamform_tc_kernel<64, 4>}};
    const Kern k = kerns[N == 64][natoms - 1];
    rc = ensure_dyn_smem((const void*)k, smem);
    if (rc == DD_OK) k<<<grid, kTcThreads, smem, st>>>(q);
    cudaError_t e = cudaGetLastError();
    cudaFreeAsync(Bimg, st);
    if (rc != DD_OK) return rc;
    if (e != cudaSuccess) return fail(DD_ERR_CUDA, std::string("tcgen05 beamformer launch: ") + cudaGetErrorString(e));
    return DD_OK;
}

}  // namespace dd
