// float32 kernel with shared partial sums (SURVEY.md §8 rows a2, a4, a5, a6 for the float32 path).
//
// What is computed is eq 2.1 exactly: every output is the sum of the same
// nchans operands.  How: a float32 word holds one sample, so the thesis' loop (Alg. 1,
// one shared-memory read per add) is capped at 32 adds/clk/SM, a quarter of
// the FP32 add rate.  Here the channels are taken in groups of G = 4 or 8 (chosen per plan by a
// cost model; the text below writes G = 4).  Within a tile of KB = 64 or 128
// adjacent (sorted) trials the relative delays of a group,
//     r_k(d) = s(d, c0+k) - s(d, c0),  k = 1..3,
// take only a few distinct values ("patterns": 3-7 per tile on the BASELINE.json workloads,
// because adjacent channels and adjacent trials differ by a fraction of a sample).  Per group a
// block therefore
//   1. has the four channel vectors (eq 2.14) in shared memory, copied there by the
//      TMA engine (cp.async.bulk + mbarrier, three stages ahead);
//   2. forms one row per pattern,  P[u] = ((x0[u] + x1[u+r1]) + x2[u+r2]) + x3[u+r3],  in shared
//      memory (all warps, 64 consecutive u per warp step);
//   3. adds, for every trial d and sample t of the tile, ONE word:  acc += P_{pattern(d)}[t + s(d,c0)].
// Step 3 costs one shared-memory word per FOUR channel-adds; step 2 adds about (patterns / KB)
// * 5/4 words per channel-add.  Descriptors (windows, patterns, per-trial row offsets) are built on
// the host at plan time from the exact delay table; nothing is approximated, and the order of
// the additions depends only on the plan (groups in ascending channel order, inside a group the
// expression above), never on the tile, so batch / streaming / one-shot results are identical.
//
// Layout of a block: 16 warps; warp w owns trials w*KW .. w*KW+KW-1 of the tile, lane l owns
// the output samples t0 + l + 32 i, i < NK (accumulators acc[KW][NK] in registers, KW * NK = 64,
// PAPER.md:958).  D is written once with 128-byte coalesced warp stores.
#include <cuda_runtime.h>

#include <algorithm>
#include <new>
#include <vector>

#include "dd_internal.h"
#include "ps_host.h"
#include "tma_ptx.cuh"

struct dd_ps_plan {
    bool ok = false;
    int ntiles = 0, ngroups = 0;
    int G = 4;                     // channels per group
    int kw = 4;                    // trials per warp (block = 16 kw trials x 32 * 64 / kw samples)
    int desc_ints = 0;             // ints per (tile, group) descriptor (multiple of 4)
    int xw = 0;                    // words per staged channel vector
    int psw = 0;                   // words of one partial-sum buffer
    size_t smem = 0;
    int32_t* d_desc = nullptr;     // device [ntiles][ngroups][desc_ints]
};

namespace dd {

namespace {

constexpr int kGMax = kPsGMax;            // channels per group: 4 or 8
constexpr int kWarps = 16;
constexpr int kThreads = 32 * kWarps;
// tile shapes: KW trials per warp x NK = 64 / KW samples per lane (64 accumulators per thread), i.e.
// 64 trials x 512 samples or 128 trials x 256 samples per block; chosen per plan by the cost model
constexpr int kAccPerLane = 64;
constexpr int kKBMax = 8 * kWarps;
constexpr int kXStages = 3;
constexpr int kMaxSmem = 200 * 1024;

// descriptor layout (ints), one per (trial tile, channel group)
constexpr int kChunk = 64;                // words of a partial-sum row formed per warp step
constexpr int kDNChunks = 0;              // kChunk-word steps of the partial-sum phase
constexpr int kDBytes = 1;                // bytes of this descriptor that are in use (multiple of 16)
constexpr int kDBase = 4;                 // [8]  first staged word of channel k, relative to t0 (multiple of 4)
constexpr int kDLen = 12;                 // [8]  words to stage (multiple of 4; 0 for a missing channel)
constexpr int kDTrial = 20;               // [KB] flat word offset of trial j's first operand in the partial sums
// kDTrial + KB:                             [nchunks][G] uint16 word offset, from the stage's first staged word, of
                                          //      the operand of lane 0 in channel k (zero pad if missing); 16-bit
                                          //      entries because a warp-uniform LDS.128 still costs four data cycles

struct PsParams {
    const float* X;
    float* D;
    const int32_t* desc;
    const int32_t* order;
    int nchans, ndm, ngroups, desc_ints, xw, psw;
    int64_t nsamp, row_valid;      // row_valid: words of a channel row that may be read (multiple of 4)
    int64_t in_stride, in_beam_stride, out_stride, out_beam_stride;
};

template <int G, int KW>
__global__ void __launch_bounds__(kThreads + 32, 1)
dd_ps_f32_kernel(const PsParams p)
{
    constexpr int NK = kAccPerLane / KW, KB = KW * kWarps, TB = 32 * NK, kDChunk = kDTrial + KB;
    extern __shared__ __align__(128) uint8_t smem_raw[];
    const int xstage = G * p.xw + kChunk;                                      // words; the last kChunk stay zero
    float* Xs = reinterpret_cast<float*>(smem_raw);                            // [kXStages][xstage]
    float* Ps = Xs + kXStages * xstage;                                        // [2][psw]
    int32_t* Ds = reinterpret_cast<int32_t*>(Ps + 2 * p.psw);                  // [kXStages][desc_ints]
    uint64_t* full = reinterpret_cast<uint64_t*>(Ds + kXStages * p.desc_ints); // [kXStages]
    uint64_t* empty = full + kXStages;                                         // [kXStages]
    uint64_t* ready = empty + kXStages;                                        // [2] partial sums complete
    uint64_t* freeb = ready + 2;                                               // [2] partial sums consumed

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = blockIdx.x;                          // trial tiles fastest: neighbours share L2 lines
    const int64_t t0 = (int64_t)blockIdx.y * TB;
    const int beam = blockIdx.z;
    const int ng = p.ngroups;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kXStages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], kWarps);
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(&ready[b], kWarps);
            mbar_init(&freeb[b], kWarps);
        }
        mbar_fence_init();
    }
    if (threadIdx.x < kXStages * kChunk)
        Xs[(threadIdx.x / kChunk) * xstage + G * p.xw + (threadIdx.x % kChunk)] = 0.0f;
    __syncthreads();

    if (warp == kWarps) {
        // ---------------------------------------------------------------- producer warp
        // lane k < G stages channel k of the group, lane G the descriptor; a stage is refilled as
        // soon as all 16 consumer warps have released it.
        const int32_t* gdesc = p.desc + (int64_t)tile * ng * p.desc_ints;
        const float* Xb = p.X + (int64_t)beam * p.in_beam_stride + t0;
        for (int g = 0; g < ng; ++g) {
            const int st = g % kXStages;
            const int32_t* dg = gdesc + (int64_t)g * p.desc_ints;
            const int hv = lane < kDTrial ? __ldg(dg + lane) : 0;           // header words
            const int base = __shfl_sync(0xffffffffu, hv, kDBase + (lane & 7));
            int len = __shfl_sync(0xffffffffu, hv, kDLen + (lane & 7));
            const int dbytes = __shfl_sync(0xffffffffu, hv, kDBytes);
            // the last time tile must not read past the row
            len = (int)max((int64_t)0, min((int64_t)len, p.row_valid - (t0 + base)));
            const uint32_t bytes = lane < G ? (uint32_t)len * 4u : (lane == G ? (uint32_t)dbytes : 0u);
            uint32_t total = bytes;
#pragma unroll
            for (int o = 8; o >= 1; o >>= 1) total += __shfl_xor_sync(0xffffffffu, total, o);   // lanes 0..15
            if (g >= kXStages) mbar_wait(&empty[st], ((g / kXStages) - 1) & 1);
            if (lane == 0) mbar_arrive_expect_tx(&full[st], total);
            __syncwarp();
            if (lane < G) {
                if (len > 0)
                    bulk_load(Xs + st * xstage + lane * p.xw, Xb + (int64_t)(g * G + lane) * p.in_stride + base,
                              bytes, &full[st]);
            } else if (lane == G) {
                bulk_load(Ds + st * p.desc_ints, dg, bytes, &full[st]);
            }
        }
        return;
    }

    // -------------------------------------------------------------------- consumer warps
    // Step 2: the pattern rows of group g into partial-sum buffer `buf`; a warp step forms kChunk
    // consecutive words (lane l: words l and l + 32) from one descriptor entry of G byte offsets.
    auto pre = [&](int st, int buf) {
        const int32_t* ds = Ds + st * p.desc_ints;
        const uint32_t xa = smem_u32(Xs + st * xstage) + lane * 4;
        float* ps = Ps + buf * p.psw + lane;
        const int nchunks = ds[kDNChunks];
        const uint32_t* ct = reinterpret_cast<const uint32_t*>(ds + kDChunk);
        for (int c = warp; c < nchunks; c += kWarps) {
            uint32_t pk[G / 2];
            if (G == 4) {
                const uint2 v = *reinterpret_cast<const uint2*>(ct + c * 2);
                pk[0] = v.x; pk[1] = v.y;
            } else {
                const uint4 v = *reinterpret_cast<const uint4*>(ct + c * 4);
                pk[0] = v.x; pk[1] = v.y; pk[G / 2 - 2] = v.z; pk[G / 2 - 1] = v.w;
            }
            int o[G];
#pragma unroll
            for (int q = 0; q < G / 2; ++q) {
                o[2 * q] = (int)(pk[q] & 0xffffu) * 4;
                o[2 * q + 1] = (int)(pk[q] >> 16) * 4;
            }
            float lo[G], hi[G];
#pragma unroll
            for (int k = 0; k < G; ++k) {
                lo[k] = lds_f32(xa + o[k]);
                hi[k] = lds_f32(xa + o[k] + 128);
            }
            float slo = lo[0], shi = hi[0];
#pragma unroll
            for (int k = 1; k < G; ++k) { slo += lo[k]; shi += hi[k]; }
            ps[c * kChunk] = slo;
            ps[c * kChunk + 32] = shi;
        }
    };

    float acc[KW][NK];
#pragma unroll
    for (int j = 0; j < KW; ++j)
#pragma unroll
        for (int i = 0; i < NK; ++i) acc[j][i] = 0.0f;

    // Warps synchronise through split-phase barriers instead of a block barrier: ready[b] completes
    // when all 16 warps have written their part of partial-sum buffer b, freeb[b] when all have
    // consumed it; a warp only waits if another one is a whole phase behind.
    mbar_wait(&full[0], 0);
    pre(0, 0);
    __syncwarp();
    if (lane == 0) mbar_arrive(&ready[0]);

    int st = 0, sn = 1 % kXStages, phn = kXStages == 1 ? 1 : 0;
    for (int g = 0; g < ng; ++g) {
        const int b = g & 1;
        if (g + 1 < ng) {
            mbar_wait(&full[sn], phn);
            if (g >= 1) mbar_wait(&freeb[b ^ 1], ((g - 1) >> 1) & 1);      // step 3 of g-1 is done everywhere
            pre(sn, b ^ 1);
            __syncwarp();
            if (lane == 0) mbar_arrive(&ready[b ^ 1]);
        }
        // Step 3: one word per trial, sample and group
        int tro[KW];
#pragma unroll
        for (int q = 0; q < KW / 4; ++q) {
            const int4 tr = *reinterpret_cast<const int4*>(Ds + st * p.desc_ints + kDTrial + warp * KW + 4 * q);
            tro[4 * q] = tr.x; tro[4 * q + 1] = tr.y; tro[4 * q + 2] = tr.z; tro[4 * q + 3] = tr.w;
        }
        const float* ps = Ps + b * p.psw + lane;
        mbar_wait(&ready[b], (g >> 1) & 1);                                // step 2 of g is done everywhere
#pragma unroll
        for (int j = 0; j < KW; ++j) {
            const float* r = ps + tro[j];
#pragma unroll
            for (int i = 0; i < NK; ++i) acc[j][i] += r[32 * i];
        }
        __syncwarp();
        if (lane == 0) {
            mbar_arrive(&freeb[b]);
            mbar_arrive(&empty[st]);                     // stage st (vectors and descriptor) may be refilled
        }
        st = sn;
        if (++sn == kXStages) { sn = 0; phn ^= 1; }
    }

    float* Db = p.D + (int64_t)beam * p.out_beam_stride;
#pragma unroll
    for (int j = 0; j < KW; ++j) {
        const int d = tile * KB + warp * KW + j;
        if (d < p.ndm) {
            float* drow = Db + (int64_t)__ldg(p.order + d) * p.out_stride + t0 + lane;
#pragma unroll
            for (int i = 0; i < NK; ++i)
                if (t0 + lane + 32 * i < p.nsamp) drow[32 * i] = acc[j][i];
        }
    }
}

// 2-D copy of the valid part of every row into a 16-byte aligned, padded workspace (used when the
// caller's X is not 16-byte aligned or its strides are not multiples of four elements)
__global__ void __launch_bounds__(256)
dd_repitch_f32(const float* __restrict__ X, float* __restrict__ W, int nchans, int64_t rowlen, int64_t in_stride,
               int64_t in_beam_stride, int64_t wpitch)
{
    const int64_t row = blockIdx.x;                       // rows on grid.x: no 65535 limit on nbeams * nchans
    const float* src = X + (row / nchans) * in_beam_stride + (row % nchans) * in_stride;
    float* dst = W + row * wpitch;
    for (int64_t i = (int64_t)blockIdx.y * blockDim.x + threadIdx.x; i < wpitch; i += (int64_t)gridDim.y * blockDim.x)
        dst[i] = i < rowlen ? src[i] : 0.0f;
}

}  // namespace

namespace {

typedef void (*PsKernel)(const PsParams);
PsKernel ps_kernel_for(int G, int kw)
{
    if (kw == 8) return G == 8 ? dd_ps_f32_kernel<8, 8> : dd_ps_f32_kernel<4, 8>;
    return G == 8 ? dd_ps_f32_kernel<8, 4> : dd_ps_f32_kernel<4, 4>;
}

struct PsShape { bool fits = false; int64_t psw = 0, xw = 0; int desc_ints = 0; size_t smem = 0; double cost = 0; };

// Shared-memory need and modelled shared-memory wavefronts per output tile for group size G:
// step 3 costs KB * NK per group, step 2 (2 G + 2 + G / 2) per kChunk words of pattern rows.
PsShape shape_for(const HostTable& h, int G, int kw)
{
    PsShape o;
    const int kKB = kw * kWarps, kNK = kAccPerLane / kw, kTB = 32 * kNK, kDChunk = kDTrial + kKB;
    const int ntiles = (h.ndm + kKB - 1) / kKB, ngroups = (h.nchans + G - 1) / G;
    const int64_t spread = max_tile_spread(h, kKB);
    o.xw = (kTB + spread + 3 + 3) / 4 * 4 + kChunk;
    const int workers = ps_workers(ntiles);
    std::vector<int64_t> wpsw(workers, 0), wchunks(workers, 0);
    ps_parallel_tiles(ntiles, workers, [&](int tb, int te, int wk) {
        std::vector<PsRow> rows;
        int slot[kKBMax];
        for (int tile = tb; tile < te; ++tile)
            for (int g = 0; g < ngroups; ++g) {
                ps_classify(h, G, kKB, tile, g, rows, slot);
                int64_t w = 0;
                for (const PsRow& r : rows) w += ((int64_t)r.umax - r.umin + kTB + kChunk - 1) / kChunk * kChunk;
                wpsw[wk] = std::max(wpsw[wk], w);
                wchunks[wk] += w / kChunk;
            }
    });
    int64_t chunks = 0;
    for (int wk = 0; wk < workers; ++wk) {
        o.psw = std::max(o.psw, wpsw[wk]);
        chunks += wchunks[wk];
    }
    o.desc_ints = (kDChunk + (G / 2) * (int)(o.psw / kChunk) + 3) / 4 * 4;
    o.smem = (size_t)kXStages * (G * o.xw + kChunk) * 4 + (size_t)2 * o.psw * 4 +
             (size_t)kXStages * o.desc_ints * 4 + (2 * kXStages + 4) * 8;
    o.fits = G * o.xw + kChunk < 65536 && o.smem <= (size_t)kMaxSmem;
    o.cost = (double)ntiles * ngroups * kKB * kNK + (double)chunks * (2 * G + 2 + G / 2);
    return o;
}

}  // namespace

int build_ps_plan(dd_plan* p)
{
    p->ps = nullptr;
    if (p->ndm == 0 || p->dtype != DD_F32) return DD_OK;
    const HostTable& h = p->host;
    const int nch = p->nchans, ndm = p->ndm;
    // group size: the cheaper of 8 and 4 by the wavefront model, among those that fit
    int G = 0, kw = 0;
    PsShape sh;
    for (int ckw : {4, 8})
        for (int cand : {8, 4}) {
            if (cand == 8 && nch < 16) continue;
            if (ckw == 8 && ndm <= 64) continue;              // a 128-trial tile would be half empty
            PsShape c = shape_for(h, cand, ckw);
            if (c.fits && (G == 0 || c.cost < sh.cost)) {
                G = cand;
                kw = ckw;
                sh = c;
            }
        }
    if (G == 0) {                    // per-trial delay steps too large / too many patterns: generic kernel
        p->ps_why = "the delay patterns of a 64-trial tile do not fit shared memory (per-trial delay steps too coarse)";
        return DD_OK;
    }
    const int kKB = kw * kWarps, kNK = kAccPerLane / kw, kTB = 32 * kNK, kDChunk = kDTrial + kKB;
    (void)kNK;
    const int ntiles = (ndm + kKB - 1) / kKB, ngroups = (nch + G - 1) / G;
    const int desc_ints = sh.desc_ints;

    dd_ps_plan* t = new (std::nothrow) dd_ps_plan;
    if (!t) return fail(DD_ERR_NOMEM, "ps plan allocation failed");
    p->ps = t;
    t->G = G;
    t->kw = kw;
    t->ntiles = ntiles;
    t->ngroups = ngroups;
    t->desc_ints = desc_ints;
    t->xw = (int)sh.xw;
    t->psw = (int)sh.psw;
    t->smem = sh.smem;

    std::vector<int32_t> desc;
    try {
        desc.assign((size_t)ntiles * ngroups * desc_ints, 0);
    } catch (const std::bad_alloc&) {
        destroy_ps_plan(p);
        return fail(DD_ERR_NOMEM, "ps descriptor allocation failed");
    }
    const int zero_pad = G * t->xw;                       // word offset of the stage's kChunk zero words
    bool bounds_ok = true;                                // every shared-memory offset written below is in range
    const int workers = ps_workers(ntiles);
    std::vector<char> wok(workers, 1);
    ps_parallel_tiles(ntiles, workers, [&](int tb, int te, int wk) {
    std::vector<PsRow> rows;
    int slot[kKBMax];
    std::vector<int> rowbase;
    bool bounds_ok = true;
    for (int tile = tb; tile < te; ++tile)
        for (int g = 0; g < ngroups; ++g) {
            ps_classify(h, G, kKB, tile, g, rows, slot);
            int32_t* ds = &desc[((size_t)tile * ngroups + g) * desc_ints];
            const int c0 = g * G, nk = std::min(G, nch - c0);
            const int dfirst = tile * kKB, dlast = std::min(tile * kKB + kKB, ndm) - 1;
            int base[kGMax] = {0, 0, 0, 0, 0, 0, 0, 0};
            for (int k = 0; k < nk; ++k) {
                const int smin = h.shift[(size_t)dfirst * nch + c0 + k], smax = h.shift[(size_t)dlast * nch + c0 + k];
                base[k] = smin & ~3;
                ds[kDBase + k] = base[k];
                ds[kDLen + k] = (smax + kTB - base[k] + 3) / 4 * 4;
            }
            int flat = 0;
            rowbase.assign(rows.size(), 0);
            for (size_t r = 0; r < rows.size(); ++r) {
                rowbase[r] = flat;
                const int ulen = rows[r].umax - rows[r].umin + kTB;
                // word e of the flat partial-sum buffer (rowbase <= e < rowbase + ulen) is
                // u = umin + (e - rowbase); channel k supplies x_k[u + r_k], staged at word
                // (u + r_k - base_k) of its vector
                for (int c = 0; c < (ulen + kChunk - 1) / kChunk; ++c) {
                    uint16_t* ce = reinterpret_cast<uint16_t*>(ds + kDChunk) + G * (flat / kChunk + c);
                    for (int k = 0; k < G; ++k) {
                        const int rk = k == 0 ? 0 : rows[r].key[k - 1];
                        const int off = k < nk ? k * t->xw + rows[r].umin + kChunk * c + rk - base[k] : zero_pad;
                        // every lane's two reads (words off + l and off + l + 32) stay inside the stage
                        bounds_ok = bounds_ok && off >= 0 && off + kChunk <= G * t->xw + kChunk;
                        ce[k] = (uint16_t)off;
                    }
                }
                flat += (ulen + kChunk - 1) / kChunk * kChunk;
            }
            ds[kDNChunks] = flat / kChunk;
            ds[kDBytes] = (4 * kDChunk + 2 * G * (flat / kChunk) + 15) / 16 * 16;
            for (int j = 0; j < kKB; ++j) {
                const int d = std::min(tile * kKB + j, ndm - 1);
                const int s0 = h.shift[(size_t)d * nch + c0];
                ds[kDTrial + j] = rowbase[slot[j]] + (s0 - rows[slot[j]].umin);
                bounds_ok = bounds_ok && ds[kDTrial + j] >= 0 && ds[kDTrial + j] + kTB <= t->psw;
            }
        }
    wok[wk] = bounds_ok;
    });
    for (int wk = 0; wk < workers; ++wk) bounds_ok = bounds_ok && wok[wk];
    if (!bounds_ok) {                                     // never expected; the plan stays unusable (generic kernel)
        p->ps_why = "descriptor bounds check failed";
        return DD_OK;
    }
    cudaError_t e = cudaMalloc(&t->d_desc, desc.size() * sizeof(int32_t));
    if (e != cudaSuccess) {
        cudaGetLastError();
        destroy_ps_plan(p);
        return fail(DD_ERR_NOMEM, std::string("ps descriptor table: ") + cudaGetErrorString(e));
    }
    e = cudaMemcpy(t->d_desc, desc.data(), desc.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        destroy_ps_plan(p);
        return fail(DD_ERR_CUDA, std::string("ps descriptor upload: ") + cudaGetErrorString(e));
    }
    t->ok = true;
    return DD_OK;
}

void destroy_ps_plan(dd_plan* p)
{
    if (!p->ps) return;
    if (p->ps->d_desc) cudaFree(p->ps->d_desc);
    delete p->ps;
    p->ps = nullptr;
}

bool ps_plan_usable(const dd_plan* p) { return p->ps && p->ps->ok; }

static bool ps_direct(const ExecArgs& a)
{
    return (((uintptr_t)a.X & 15) == 0) && (a.in_stride & 3) == 0 && (a.nbeams == 1 || (a.in_beam_stride & 3) == 0);
}

bool ps_args_ok(const dd_plan* p, const ExecArgs& a)
{
    if (!ps_plan_usable(p)) return false;
    const int kTB = 32 * kAccPerLane / p->ps->kw;
    if ((a.nsamp_out + kTB - 1) / kTB > 65535 || a.nbeams > 65535) return false;
    if (!ps_direct(a) && (int64_t)a.nbeams * p->nchans > 2147483647LL) return false;   // grid.x of the re-pitch copy
    return true;
}

int ps_launches(const dd_plan* p, const ExecArgs& a) { return ps_direct(a) ? 1 : 2; }

std::string ps_describe(const dd_plan* p)
{
    const dd_ps_plan* t = p->ps;
    return "partial-sum kernel dd_ps_f32_kernel<G=" + std::to_string(t->G) + ", KW=" + std::to_string(t->kw) + ">: " +
           std::to_string(16 * t->kw) + " trials x " + std::to_string(32 * kAccPerLane / t->kw) +
           " samples per block, " + std::to_string(t->smem) + " B shared memory";
}

int launch_ps(const dd_plan* p, const ExecArgs& a)
{
    const dd_ps_plan* t = p->ps;
    cudaStream_t st = (cudaStream_t)a.stream;
    const int64_t rowlen = a.nsamp_out + p->host.maxshift;
    PsParams q;
    q.X = (const float*)a.X;
    q.in_stride = a.in_stride;
    q.in_beam_stride = a.in_beam_stride;
    q.row_valid = (rowlen + 3) / 4 * 4;
    float* W = nullptr;
    if (!ps_direct(a)) {
        const int64_t wpitch = (rowlen + 3) / 4 * 4;
        const int64_t nrows = (int64_t)a.nbeams * p->nchans;
        int wrc = workspace_alloc((void**)&W, (size_t)(nrows * wpitch) * sizeof(float), a.stream);
        if (wrc != DD_OK) return wrc;
        dim3 grid((unsigned)nrows, (unsigned)std::min<int64_t>((wpitch + 255) / 256, 64));
        dd_repitch_f32<<<grid, 256, 0, st>>>((const float*)a.X, W, p->nchans, rowlen, a.in_stride, a.in_beam_stride,
                                             wpitch);
        q.X = W;
        q.in_stride = wpitch;
        q.in_beam_stride = (int64_t)p->nchans * wpitch;
    }
    q.D = (float*)a.D;
    q.desc = t->d_desc;
    q.order = a.d_order;
    q.nchans = p->nchans;
    q.ndm = p->ndm;
    q.ngroups = t->ngroups;
    q.desc_ints = t->desc_ints;
    q.xw = t->xw;
    q.psw = t->psw;
    q.nsamp = a.nsamp_out;
    q.out_stride = a.out_stride;
    q.out_beam_stride = a.out_beam_stride;
    const int kTB = 32 * kAccPerLane / t->kw;
    dim3 grid((unsigned)t->ntiles, (unsigned)((a.nsamp_out + kTB - 1) / kTB), (unsigned)a.nbeams);
    int rc = ensure_dyn_smem((const void*)ps_kernel_for(t->G, t->kw), t->smem);
    if (rc != DD_OK) {
        if (W) cudaFreeAsync(W, st);
        return rc;
    }
    ps_kernel_for(t->G, t->kw)<<<grid, kThreads + 32, t->smem, st>>>(q);
    cudaError_t e = cudaGetLastError();
    if (W) cudaFreeAsync(W, st);
    if (e != cudaSuccess) return fail(DD_ERR_CUDA, std::string("ps f32 launch: ") + cudaGetErrorString(e));
    return DD_OK;
}

}  // namespace dd
