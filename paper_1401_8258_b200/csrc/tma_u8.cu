// TMA-staged uint8 -> int32 kernel (SURVEY.md §8 rows a2-a5 for the uint8 path).
//
// What is computed is eq 2.1 exactly; how it is computed differs from the
// thesis' Alg. 1 in the three places where that design is bound on sm_100a:
//
//  a2 staging   A block owns kKB = 64 consecutive (sorted) trials x kTB = 1024 output samples.
//               For every channel the "channel vector" X[c][t0+s(d0,c) .. +1024+spread) (eq 2.14,
//               PAPER.md:945) is brought into shared memory by the TMA engine (cp.async.bulk,
//               completion on an mbarrier) -- no SM instruction touches it.  The row start
//               t0+s(d0,c) has arbitrary byte alignment (PAPER.md:986 notes the misaligned loads)
//               while bulk copies need 16-byte aligned sources (a byte-granular tensor-map
//               coordinate faults on sm_100a: measured), so a small HBM-bound front-end kernel
//               first writes four byte-shifted copies W_r[i] = X[i + r], r = 0..3, into a padded
//               workspace.  A block stages, per channel, the 16-byte aligned window of each W_r;
//               every trial then reads ALIGNED 32-bit words whatever its delay:
//               copy (a & 3), word (a >> 2), a = (t0+s(d0,c)) mod 16 + s(d,c) - s(d0,c).
//  a3/a4 unpack + accumulate   A 32-bit word w carries four samples b0..b3.  Per word the SM
//               issues one LDS and three arithmetic instructions for FOUR sample-adds (Alg. 1:
//               1 + 2 + 1 per ONE):  A += w & 0x00ff00ff  (LOP3 + add: b0 and b2 in 16-bit lanes)
//               and  C = hi32(w * 2^24) + C  (one IMAD.HI.U32: C += w >> 8 = b1 + 2^8 b2 + 2^16 b3).
//               After n <= 256 channels  sum b0 = A & 0xffff,  sum b2 = A >> 16,  and
//               C - 2^8 sum b2 = sum b1 + 2^16 sum b3  (C <= 65280 * 65793 < 2^32), so all four
//               sums are recovered exactly; they are flushed into the int32 output every
//               kFlush = 256 channels.
//  a5 store     The flush is a 16-byte read-modify-write of D (plain store for the first one); a
//               block's D tile (256 KB) stays in L2 between flushes.
//
// Channels are added in the order c = 0,1,2,... for every output element; integer arithmetic,
// so the result is exact and independent of tiling.
//
// Roofline: 4 issue slots per 4 sample-adds -> the issue rate (128 thread
// instructions/clk/SM) allows 128 sample-adds/clk/SM, the same as the add roofline; the ALU and
// FMA pipes (64 lanes/clk/SM each, measured) carry 2 and 1-2 of the 4 instructions.
#include <cuda_runtime.h>

#include <algorithm>
#include <new>

#include "dd_internal.h"

struct dd_tma_plan {
    bool u8_ok = false;
    int ny = 0;                    // bytes staged per byte-shifted copy and channel, in units of 256
    int ndm_pad = 0;               // row pitch of d_shift_t (multiple of kKB)
    int32_t* d_shift_t = nullptr;  // device [nchans][ndm_pad]: s(d,c), trial index fastest, sorted DMs
};

namespace dd {

namespace {

constexpr int kConsumerWarps = 16;
constexpr int kThreads = 32 * kConsumerWarps;         // 512: 128 registers per thread, one block per SM
constexpr int kKW = 4;                                // trials per consumer warp
constexpr int kKB = kKW * kConsumerWarps;             // trials per block
constexpr int kNK = 8;                                // 32-bit words per lane (lane-interleaved)
constexpr int kTB = 32 * 4 * kNK;                     // output samples per block
constexpr int kCH = 4;                                // channels per pipeline stage
constexpr int kStages = 8;
constexpr int kLead = kStages - 1;                    // groups staged ahead (as early as a stage can be free)
constexpr int kMust = 3;                              // ... and at the latest this many groups ahead
constexpr int kFlush = 256;                           // 256 * 255 < 65536
constexpr int kMaxNY = 8;
constexpr int kBoxW = 256;                            // granule of the staged window length (bytes)

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!done);
}
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

struct U8Params {
    const uint8_t* W;              // workspace: four byte-shifted copies, [4][nbeams*nchans][wpitch]
    int64_t wcopy;                 // bytes between the copies
    int64_t wpitch;                // bytes between channel rows of a copy (multiple of 128)
    int32_t* D;
    const int32_t* shift_t;        // [nchans][ndm_pad]
    const int32_t* order;
    int nchans, ndm, ndm_pad, ny;
    int64_t nsamp, out_stride, out_beam_stride;
};

// Front end (row a3): W_r[row][i] = X[row][i + r] for r = 0..3.  One thread per output word.
__global__ void __launch_bounds__(256)
dd_shift_copies_u8(const uint8_t* __restrict__ X, uint8_t* __restrict__ W, int64_t wcopy, int64_t wpitch,
                   int nchans, int64_t rowlen, int64_t in_stride, int64_t in_beam_stride)
{
    const int64_t row = blockIdx.y;                                   // beam * nchans + channel
    const uint8_t* src = X + (row / nchans) * in_beam_stride + (row % nchans) * in_stride;
    const int sh = (int)((uintptr_t)src & 3);
    const uint32_t* srcw = reinterpret_cast<const uint32_t*>(src - sh);   // aligned words covering the row
    const int64_t nwords = (rowlen + 3) >> 2;
    const int64_t lastw = (sh + rowlen - 1) >> 2;                     // last aligned word holding a valid byte
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nwords; i += (int64_t)gridDim.x * blockDim.x) {
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

// The 8 lane-interleaved words (32 samples) of one channel that one trial needs.
__device__ __forceinline__ void load_words(uint32_t (&w)[kNK], uint32_t saddr)
{
#pragma unroll
    for (int k = 0; k < kNK; ++k)
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(w[k]) : "r"(saddr + k * 128));
}
// Adds them into the accumulators of that trial: A holds b0,b2 in 16-bit lanes, C the running
// sum of w >> 8 (see the header).
__device__ __forceinline__ void add_words(uint32_t (&A)[kNK], uint32_t (&C)[kNK], const uint32_t (&w)[kNK])
{
#pragma unroll
    for (int k = 0; k < kNK; ++k) {
        A[k] += w[k] & 0x00ff00ffu;
        asm("mad.hi.u32 %0, %1, 0x01000000, %0;" : "+r"(C[k]) : "r"(w[k]));
    }
}
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity)
{
    uint32_t done;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return done != 0;
}

__global__ void __launch_bounds__(kThreads, 1)
dd_tma_u8_kernel(const U8Params p)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const int copy_pitch = p.ny * kBoxW;                  // bytes of one byte-shifted copy
    const int chan_pitch = 4 * copy_pitch;
    const int stage_pitch = kCH * chan_pitch;
    uint8_t* rows = smem;                                                     // [kStages][kCH][4][ny*256]
    int32_t* offs = reinterpret_cast<int32_t*>(smem + kStages * stage_pitch); // [kStages][16 warps][kCH][kKW]
    uint64_t* full = reinterpret_cast<uint64_t*>(offs + kStages * kCH * kKB);
    uint64_t* empty = full + kStages;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int d0 = blockIdx.x * kKB;                      // trial tiles fastest: neighbouring blocks
    const int64_t t0 = (int64_t)blockIdx.y * kTB;         // re-read nearly the same rows through L2
    const int beam = blockIdx.z;
    const int ngroups = (p.nchans + kCH - 1) / kCH;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], kConsumerWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    // Producer role, taken in turn by every warp (group gp is staged by warp gp mod 16, kLead
    // groups ahead of its use): per channel the lanes write the trials' read offsets, then lane 0
    // arms the stage's mbarrier and issues the four bulk copies.
    const uint8_t* wrow0 = p.W + (int64_t)beam * p.nchans * p.wpitch + t0;
    auto produce = [&](int gp) {
        const int st = gp % kStages;
        const int nch = min(kCH, p.nchans - gp * kCH);
        int s0v[kCH];
#pragma unroll
        for (int ch = 0; ch < kCH; ++ch) {
            s0v[ch] = 0;
            if (ch < nch) {
                const int c = gp * kCH + ch;
                const int32_t* trow = p.shift_t + (int64_t)c * p.ndm_pad + d0;   // padded to whole tiles
                int s[kKB / 32];
#pragma unroll
                for (int q = 0; q < kKB / 32; ++q) s[q] = __ldg(trow + lane + 32 * q);
                const int s0 = __shfl_sync(0xffffffffu, s[0], 0);
#pragma unroll
                for (int q = 0; q < kKB / 32; ++q) {
                    const int a = (s0 & 15) + s[q] - s0;                // t0 is a multiple of 16
                    const int dl = lane + 32 * q;                       // trial within the tile
                    offs[((st * kConsumerWarps + dl / kKW) * kCH + ch) * kKW + dl % kKW] =
                        (a & 3) * copy_pitch + (a & ~3);
                }
                s0v[ch] = s0;
            }
        }
        __syncwarp();
        if (lane == 0) {
            mbar_arrive_expect_tx(&full[st], (uint32_t)(nch * chan_pitch));
#pragma unroll
            for (int ch = 0; ch < kCH; ++ch) {
                if (ch < nch) {
                    const uint8_t* src = wrow0 + (int64_t)(gp * kCH + ch) * p.wpitch + (s0v[ch] & ~15);
                    uint8_t* dst = rows + st * stage_pitch + ch * chan_pitch;
#pragma unroll
                    for (int r = 0; r < 4; ++r)
                        bulk_load(dst + r * copy_pitch, src + r * p.wcopy, (uint32_t)copy_pitch, &full[st]);
                }
            }
        }
        __syncwarp();
    };
    // A warp whose turn it is stages the group as soon as the stage's previous users have all
    // released it; until then it keeps consuming and polls (a blocked producer would stall every
    // other warp one group later).  kMust groups before the data is needed it waits.
    int pending = -1;
    auto try_produce = [&](bool must) {
        const int st = pending % kStages;
        if (pending >= kStages) {
            const uint32_t par = ((pending / kStages) - 1) & 1;
            if (must) mbar_wait(&empty[st], par);
            else if (!mbar_test(&empty[st], par)) return;
        }
        produce(pending);
        pending = -1;
    };
    for (int gp = 0; gp < kLead && gp < ngroups; ++gp)
        if (gp % kConsumerWarps == warp) produce(gp);

    // -------------------------------------------------------------------- consumer warps
    uint32_t A[kKW][kNK], C[kKW][kNK];
#pragma unroll
    for (int j = 0; j < kKW; ++j)
#pragma unroll
        for (int k = 0; k < kNK; ++k) A[j][k] = C[j][k] = 0;

    int32_t* Db = p.D + (int64_t)beam * p.out_beam_stride;
    int nflush = 0;

    auto flush = [&]() {
#pragma unroll
        for (int j = 0; j < kKW; ++j) {
            const int d = d0 + warp * kKW + j;
            if (d < p.ndm) {
                int32_t* drow = Db + (int64_t)__ldg(p.order + d) * p.out_stride;
#pragma unroll
                for (int k = 0; k < kNK; ++k) {
                    const int64_t t = t0 + 4 * (lane + 32 * k);
                    const uint32_t b0 = A[j][k] & 0xffffu, b2 = A[j][k] >> 16;
                    const uint32_t r = C[j][k] - (b2 << 8);               // sum b1 + 2^16 sum b3
                    int4 v = make_int4((int)b0, (int)(r & 0xffffu), (int)b2, (int)(r >> 16));
                    if (t + 3 < p.nsamp) {
                        int4* q = reinterpret_cast<int4*>(drow + t);
                        if (nflush) {
                            const int4 old = __ldcg(q);
                            v.x += old.x; v.y += old.y; v.z += old.z; v.w += old.w;
                        }
                        *q = v;
                    } else {
                        const int vv[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            if (t + e < p.nsamp) drow[t + e] = (nflush ? __ldcg(drow + t + e) : 0) + vv[e];
                    }
                }
            }
#pragma unroll
            for (int k = 0; k < kNK; ++k) A[j][k] = C[j][k] = 0;
        }
        ++nflush;
    };

    auto channel = [&](int st, int ch, const int4 o4) {
        const uint32_t base = smem_u32(rows + st * stage_pitch + ch * chan_pitch + lane * 4);
        // loads of the next trial are in flight while the current one is unpacked and added
        uint32_t wa[kNK], wb[kNK];
        load_words(wa, base + o4.x);
        load_words(wb, base + o4.y);
        add_words(A[0], C[0], wa);
        load_words(wa, base + o4.z);
        add_words(A[1], C[1], wb);
        load_words(wb, base + o4.w);
        add_words(A[2], C[2], wa);
        add_words(A[3], C[3], wb);
    };

    for (int g = 0; g < ngroups; ++g) {
        if (g + kLead < ngroups && (g + kLead) % kConsumerWarps == warp) pending = g + kLead;
        if (pending >= 0) try_produce(pending - g <= kMust);
        const int st = g % kStages;
        mbar_wait(&full[st], (g / kStages) & 1);
        const int4* o = reinterpret_cast<const int4*>(offs + (st * kConsumerWarps + warp) * kCH * kKW);
        if (g * kCH + kCH <= p.nchans) {
            const int4 o0 = o[0], o1 = o[1], o2 = o[2], o3 = o[3];
            channel(st, 0, o0);
            channel(st, 1, o1);
            if (pending >= 0) try_produce(false);
            channel(st, 2, o2);
            channel(st, 3, o3);
        } else {
            for (int ch = 0; ch < p.nchans - g * kCH; ++ch) channel(st, ch, o[ch]);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[st]);
        const int c1 = (g + 1) * kCH;                                   // kFlush is a multiple of kCH
        if ((c1 & (kFlush - 1)) == 0 && c1 < p.nchans) flush();
    }
    flush();
}

size_t u8_smem_bytes(int ny)
{
    return (size_t)kStages * kCH * 4 * ny * kBoxW + (size_t)kStages * kCH * kKB * 4 + 2 * kStages * 8;
}

}  // namespace

int build_tma_plan(dd_plan* p)
{
    p->tma = nullptr;
    if (p->ndm == 0 || p->dtype != DD_U8) return DD_OK;
    const int64_t spread = max_tile_spread(p->host, kKB);
    const int ny = (int)((15 + spread + kTB + kBoxW - 1) / kBoxW);
    if (ny > kMaxNY) return DD_OK;                       // per-trial steps too large: generic kernel
    dd_tma_plan* t = new (std::nothrow) dd_tma_plan;
    if (!t) return fail(DD_ERR_NOMEM, "tma plan allocation failed");
    p->tma = t;
    t->ny = ny;
    // transposed delay table, trial index fastest, padded to whole tiles with the last trial
    t->ndm_pad = (p->ndm + kKB - 1) / kKB * kKB;
    std::vector<int32_t> tt((size_t)p->nchans * t->ndm_pad);
    for (int c = 0; c < p->nchans; ++c)
        for (int d = 0; d < t->ndm_pad; ++d)
            tt[(size_t)c * t->ndm_pad + d] = p->host.shift[(size_t)std::min(d, p->ndm - 1) * p->nchans + c];
    cudaError_t e = cudaMalloc(&t->d_shift_t, tt.size() * sizeof(int32_t));
    if (e != cudaSuccess) {
        cudaGetLastError();
        destroy_tma_plan(p);
        return fail(DD_ERR_NOMEM, std::string("device table allocation: ") + cudaGetErrorString(e));
    }
    e = cudaMemcpy(t->d_shift_t, tt.data(), tt.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        destroy_tma_plan(p);
        return fail(DD_ERR_CUDA, std::string("table upload: ") + cudaGetErrorString(e));
    }
    e = cudaFuncSetAttribute(dd_tma_u8_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)u8_smem_bytes(ny));
    if (e != cudaSuccess) {
        cudaGetLastError();
        destroy_tma_plan(p);
        return DD_OK;
    }
    t->u8_ok = true;
    return DD_OK;
}

void destroy_tma_plan(dd_plan* p)
{
    if (!p->tma) return;
    if (p->tma->d_shift_t) cudaFree(p->tma->d_shift_t);
    delete p->tma;
    p->tma = nullptr;
}

bool tma_plan_usable(const dd_plan* p) { return p->tma && p->tma->u8_ok; }

bool tma_args_ok(const dd_plan* p, const ExecArgs& a)
{
    if (!tma_plan_usable(p)) return false;
    // 16-byte read-modify-write of D
    if (((uintptr_t)a.D & 15) || (a.out_stride & 3) || (a.nbeams > 1 && (a.out_beam_stride & 3))) return false;
    if ((a.nsamp_out + kTB - 1) / kTB > 65535 || a.nbeams > 65535) return false;
    if ((int64_t)a.nbeams * p->nchans > 65535) return false;          // grid.y of the front end
    return true;
}

// Front end shared with ps_u8.cu: allocates (stream-ordered) and fills the four byte-shifted copies.
// Rows are padded so that the last time tile may over-read its window (the excess only feeds
// output samples >= nsamp_out, which are never stored).  The caller frees *W with cudaFreeAsync.
int make_shift_copies_u8(const dd_plan* p, const ExecArgs& a, uint8_t** W_out, int64_t* wcopy_out, int64_t* wpitch_out)
{
    cudaStream_t st = (cudaStream_t)a.stream;
    const int64_t rowlen = a.nsamp_out + p->host.maxshift;            // valid samples per channel row
    // layout [beam * nchans + channel][copy r][wcopy bytes]: the four copies of a channel are adjacent
    // rows (ps_u8.cu fetches the 16 rows of a four-channel group with one tensor copy)
    const int64_t wcopy = (rowlen + (int64_t)kMaxNY * kBoxW + 16 + 127) / 128 * 128;
    const int64_t wpitch = 4 * wcopy;
    const int64_t nrows = (int64_t)a.nbeams * p->nchans;
    uint8_t* W = nullptr;
    int rc = workspace_alloc((void**)&W, (size_t)(nrows * wpitch), a.stream);
    if (rc != DD_OK) return rc;
    const int64_t nwords = (rowlen + 3) / 4;
    dim3 grid((unsigned)std::min<int64_t>((nwords + 255) / 256, 64), (unsigned)nrows);
    dd_shift_copies_u8<<<grid, 256, 0, st>>>((const uint8_t*)a.X, W, wcopy, wpitch, p->nchans, rowlen,
                                             a.in_stride, a.in_beam_stride);
    *W_out = W;
    *wcopy_out = wcopy;
    *wpitch_out = wpitch;
    return DD_OK;
}

int launch_tma(const dd_plan* p, const ExecArgs& a)
{
    const dd_tma_plan* t = p->tma;
    cudaStream_t st = (cudaStream_t)a.stream;
    uint8_t* W = nullptr;
    int64_t wcopy = 0, wpitch = 0;
    int rc = make_shift_copies_u8(p, a, &W, &wcopy, &wpitch);
    if (rc != DD_OK) return rc;
    cudaError_t e;
    U8Params q;
    q.W = W;
    q.wcopy = wcopy;
    q.wpitch = wpitch;
    q.D = (int32_t*)a.D;
    q.shift_t = t->d_shift_t;
    q.order = a.d_order;
    q.nchans = p->nchans;
    q.ndm = p->ndm;
    q.ndm_pad = t->ndm_pad;
    q.ny = t->ny;
    q.nsamp = a.nsamp_out;
    q.out_stride = a.out_stride;
    q.out_beam_stride = a.out_beam_stride;
    dim3 grid((unsigned)((p->ndm + kKB - 1) / kKB), (unsigned)((a.nsamp_out + kTB - 1) / kTB), (unsigned)a.nbeams);
    dd_tma_u8_kernel<<<grid, kThreads, u8_smem_bytes(t->ny), st>>>(q);
    e = cudaGetLastError();
    cudaFreeAsync(W, st);
    if (e != cudaSuccess) return fail(DD_ERR_CUDA, std::string("tma u8 launch: ") + cudaGetErrorString(e));
    return DD_OK;
}

}  // namespace dd
