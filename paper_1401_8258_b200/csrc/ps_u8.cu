// uint8 -> int32 kernel with shared partial sums (SURVEY.md §8 rows a2-a6 for the uint8 path).
//
// Same idea as ps_f32.cu, same result as eq 2.1, exact integer arithmetic:
// channels are taken in groups of G = 4; within a tile of KB = 128 (or 64) adjacent (sorted) trials the relative
// delays r_k(d) = s(d,c0+k) - s(d,c0) take a handful of distinct values ("patterns"), so a block
//   1. has the channel vectors of the group in shared memory (eq 2.14): for every
//      channel the 16-byte aligned window of each of the four byte-shifted copies W_r[i] = X[i+r]
//      that the front end of tma_u8.cu writes (bulk copies need aligned sources, the window start
//      t0 + s(d0,c) is arbitrary), copied by the TMA engine three groups ahead;
//   2. forms, per pattern, the row of partial sums P[u] = x0[u] + x1[u+r1] + x2[u+r2] + x3[u+r3]
//      (<= 4*255, so 16 bits) TWICE, as 32-bit words holding (P[u], P[u+1]) for even and for odd u:
//      one aligned LDS gives four consecutive samples of a channel, two PRMT widen them into two
//      words of 16-bit lanes, adds sum the channels -> the even-u words; the odd-u words are cut
//      from those and the neighbouring lane's (one SHFL, two PRMT); warp steps overlap by one
//      lane (124 new samples per step) so that no step needs its successor;
//   3. adds ONE word per trial, per PAIR of output samples and per group:
//      acc(16-bit lanes) += P^{parity}_{pattern(d)}[(t + s(d,c0)) / 2].
// Step 3 is one shared-memory word and one integer add per EIGHT channel-sample adds (Alg. 1,
// PAPER.md:960-988, spends one word and two instructions per ONE).  The packed accumulators are
// flushed into the int32 output every kFlushGroups groups (64 * 4 * 255 < 65536) by a 16-byte
// read-modify-write that stays in L2 (plain store the first time).
//
// Layout of a block: 16 consumer warps + 1 producer warp; consumer warp w owns trials
// w*KW .. w*KW+KW-1, lane l owns output samples t0 + 2 (l + 32 i) + {0,1}, i < NK = 64 / KW.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <new>
#include <vector>

#include "dd_internal.h"
#include "ps_host.h"
#include "tma_ptx.cuh"

struct dd_psu8_plan {
    bool ok = false;
    int ntiles = 0, ngroups = 0;
    int desc_ints = 0;             // ints per (tile, group) descriptor (multiple of 4)
    int xwb = 0;                   // bytes staged per row (one byte-shifted copy of one channel; multiple of 16)
    int xstage = 0;                // bytes of one stage: 16 rows, 256 zero bytes, over-read slack
    int psw = 0;                   // words of one partial-sum buffer
    int kw = 8;                    // trials per warp (block = 16 kw trials x 64 * 64 / kw samples)
    size_t smem = 0;
    int32_t* d_desc = nullptr;     // device [ntiles][ngroups][desc_ints]
};

namespace dd {

namespace {

constexpr int kG = 4;                     // channels per group
constexpr int kWarps = 16;
constexpr int kThreads = 32 * kWarps;
// tile shapes: KW trials per warp x NK = 64 / KW sample PAIRS per lane (64 packed accumulators per
// thread): 128 trials x 512 samples per block, or 64 x 1024 for plans of at most 64 trials
constexpr int kAccPerLane = 64;
constexpr int kKBMax = 8 * kWarps;
constexpr int kXStages = 3;
constexpr int kPB = 3;                    // partial-sum buffers: step 2 may run two groups ahead of step 3
constexpr int kMaxSmem = 200 * 1024;
constexpr int kFlushGroups = 64;          // 64 groups * 4 channels * 255 = 65280 < 65536
constexpr int kChunk = 64;                // even-u words (= 128 samples) a warp step writes ...
constexpr int kStepW = 62;                // ... of which the last two are rewritten by the next step
constexpr int kCE = 4;                    // ints per step entry of the descriptor (six 16-bit fields: one 16-byte read)

// descriptor layout (ints), one per (trial tile, channel group)
constexpr int kDNChunks = 0;
constexpr int kDBytes = 1;                // bytes of this descriptor that are in use (multiple of 16)
constexpr int kDBase = 4;                 // first staged sample of the group's rows, relative to t0 (multiple of 16)
constexpr int kDTrial = 12;               // [KB / 2] uint16 x KB: word offset of trial j's first operand in the partial sums
                                          //      (the region keeps KB ints)
// kDTrial + KB:                             [nchunks][kCE]: [0..3] byte offset, from the stage's first byte, of the
                                          //      aligned word lane 0 reads in channel k (zero pad if missing);
                                          //      [4], [5] first even-u / odd-u word the step writes (even numbers)

struct PsU8Params {
    int32_t* D;
    const int32_t* desc;
    const int32_t* order;
    int nchans, ndm, ngroups, desc_ints, xwb, xstage, psw;
    int vec_ok;                    // D rows are 16-byte aligned: 16-byte read-modify-write, else element by element
    int64_t nsamp, out_stride, out_beam_stride;
};

template <int KW>
__global__ void __launch_bounds__(kThreads + 32, 1)
dd_ps_u8_kernel(const PsU8Params p, const __grid_constant__ CUtensorMap tmap)
{
    constexpr int NK = kAccPerLane / KW, KB = KW * kWarps, TB = 2 * 32 * NK, kDChunk = kDTrial + KB;
    extern __shared__ __align__(128) uint8_t smem_raw[];
    const int xstage = p.xstage;                                               // bytes: 16 rows of xwb, 256 zero bytes, slack
    uint8_t* Xs = smem_raw;                                                    // [kXStages][xstage]
    uint32_t* Ps = reinterpret_cast<uint32_t*>(Xs + kXStages * xstage);        // [kPB][psw]
    int32_t* Ds = reinterpret_cast<int32_t*>(Ps + kPB * p.psw);                // [kXStages][desc_ints]
    uint64_t* full = reinterpret_cast<uint64_t*>(Ds + kXStages * p.desc_ints); // [kXStages]
    uint64_t* empty = full + kXStages;                                         // [kXStages]
    uint64_t* ready = empty + kXStages;                                        // [kPB] partial sums complete
    uint64_t* freeb = ready + kPB;                                             // [kPB] partial sums consumed

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t xs0 = smem_u32(Xs);
    const int tile = blockIdx.x;                          // trial tiles fastest: neighbours share L2 lines
    const int64_t t0 = (int64_t)blockIdx.y * TB;
    const int beam = blockIdx.z;
    const int ng = p.ngroups;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kXStages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], kWarps);
        }
        for (int b = 0; b < kPB; ++b) {
            mbar_init(&ready[b], kWarps);
            mbar_init(&freeb[b], kWarps);
        }
        mbar_fence_init();
    }
    if (threadIdx.x < kXStages * kChunk)
        reinterpret_cast<uint32_t*>(Xs + (threadIdx.x / kChunk) * xstage + kG * 4 * p.xwb)[threadIdx.x % kChunk] = 0u;
    __syncthreads();

    if (warp == kWarps) {
        // ---------------------------------------------------------------- producer warp
        // lane 0 stages the group's channel vectors and its descriptor; a stage is refilled as soon
        // as all 16 consumer warps have released it.
        const int32_t* gdesc = p.desc + (int64_t)tile * ng * p.desc_ints;
        for (int g = 0; g < ng; ++g) {
            const int st = g % kXStages;
            const int32_t* dg = gdesc + (int64_t)g * p.desc_ints;
            const int hv = lane < kDTrial ? __ldg(dg + lane) : 0;           // header words
            const int base = __shfl_sync(0xffffffffu, hv, kDBase);
            const int dbytes = __shfl_sync(0xffffffffu, hv, kDBytes);
            if (g >= kXStages) mbar_wait(&empty[st], ((g / kXStages) - 1) & 1);
            if (lane == 0) {
                mbar_arrive_expect_tx(&full[st], (uint32_t)(4 * kG * p.xwb + dbytes));
                // one tensor copy: 16 rows (4 channels x 4 byte-shifted copies) x xwb bytes, starting at
                // sample t0 + base of every row (columns are counted in 8-byte elements)
                tensor_load_2d(Xs + st * xstage, &tmap, (int)((t0 + base) >> 3), (beam * p.nchans + g * kG) * 4,
                               &full[st]);
                bulk_load(Ds + st * p.desc_ints, dg, (uint32_t)dbytes, &full[st]);
            }
            __syncwarp();
        }
        return;
    }

    // -------------------------------------------------------------------- consumer warps
    // Step 2: a warp step forms kChunk consecutive words (128 samples) of one pattern row and parity:
    // lane l reads the aligned word with samples 4l..4l+3 of every channel and writes words 2l, 2l+1.
    // The steps of group g+1 are interleaved with step 3 of group g (below) so that their
    // shared-memory latency is covered by independent work.
    struct Words { uint32_t w0, w1, w2, w3; };
    auto pre_load = [&](uint32_t xa, const int4 o) {
        Words r;
        r.w0 = lds_u32(xa + ((uint32_t)o.x & 0xffffu)); r.w1 = lds_u32(xa + ((uint32_t)o.x >> 16));
        r.w2 = lds_u32(xa + ((uint32_t)o.y & 0xffffu)); r.w3 = lds_u32(xa + ((uint32_t)o.y >> 16));
        return r;
    };
    auto pre_store = [&](uint32_t* ps, const int4 e, const Words& r) {
        const uint2 dst = make_uint2((uint32_t)e.z & 0xffffu, (uint32_t)e.z >> 16);
        // (b0 | b1 << 16) and (b2 | b3 << 16) of each channel word, summed over the channels:
        // partial sums S0..S3 of this lane's four samples
        const uint32_t lo = __byte_perm(r.w0, 0, 0x4140) + __byte_perm(r.w1, 0, 0x4140) +
                            __byte_perm(r.w2, 0, 0x4140) + __byte_perm(r.w3, 0, 0x4140);
        const uint32_t hi = __byte_perm(r.w0, 0, 0x4342) + __byte_perm(r.w1, 0, 0x4342) +
                            __byte_perm(r.w2, 0, 0x4342) + __byte_perm(r.w3, 0, 0x4342);
        *reinterpret_cast<uint2*>(ps + dst.x + 2 * lane) = make_uint2(lo, hi);             // (S0,S1) (S2,S3)
        const uint32_t nlo = __shfl_down_sync(0xffffffffu, lo, 1);                        // next lane's (S0,S1)
        if (lane < 31)                                                                    // (S1,S2) (S3,S4)
            *reinterpret_cast<uint2*>(ps + dst.y + 2 * lane) =
                make_uint2(__byte_perm(lo, hi, 0x5432), __byte_perm(hi, nlo, 0x5432));
    };
    // all steps of the group staged in stage `st`, two in flight per warp
    auto pre = [&](int st, int buf) {
        const int32_t* ds = Ds + st * p.desc_ints;
        const uint32_t xa = xs0 + st * xstage + lane * 4;
        uint32_t* ps = Ps + buf * p.psw;
        const int nchunks = ds[kDNChunks];
        const int4* ct = reinterpret_cast<const int4*>(ds + kDChunk);
        int c = warp;
        for (; c + kWarps < nchunks; c += 2 * kWarps) {
            const int4 ea = ct[c], eb = ct[c + kWarps];
            const Words a = pre_load(xa, ea), b = pre_load(xa, eb);
            pre_store(ps, ea, a);
            pre_store(ps, eb, b);
        }
        if (c < nchunks) {
            const int4 ea = ct[c];
            pre_store(ps, ea, pre_load(xa, ea));
        }
    };

    uint32_t acc[KW][NK];
#pragma unroll
    for (int j = 0; j < KW; ++j)
#pragma unroll
        for (int i = 0; i < NK; ++i) acc[j][i] = 0u;

    int32_t* Db = p.D + (int64_t)beam * p.out_beam_stride;
    int nflush = 0;
    // lanes 2m, 2m+1 exchange halves so that every lane writes four consecutive samples
    auto flush = [&]() {
#pragma unroll
        for (int j = 0; j < KW; ++j) {
            const int d = tile * KB + warp * KW + j;
            int32_t* drow = Db + (int64_t)(d < p.ndm ? __ldg(p.order + d) : 0) * p.out_stride;
#pragma unroll
            for (int i = 0; i < NK; i += 2) {
                // this lane holds samples 2l+64i+{0,1} (acc[j][i]) and 2l+64(i+1)+{0,1} (acc[j][i+1]);
                // even lanes take both pairs of block i, odd lanes both pairs of block i+1
                const uint32_t mine = (lane & 1) ? acc[j][i + 1] : acc[j][i];
                const uint32_t give = (lane & 1) ? acc[j][i] : acc[j][i + 1];
                const uint32_t got = __shfl_xor_sync(0xffffffffu, give, 1);
                const uint32_t first = (lane & 1) ? got : mine, second = (lane & 1) ? mine : got;
                const int64_t t = t0 + 2 * (lane & ~1) + 64 * (i + (lane & 1));
                int4 v = make_int4((int)(first & 0xffffu), (int)(first >> 16), (int)(second & 0xffffu),
                                   (int)(second >> 16));
                if (d < p.ndm) {
                    if (p.vec_ok && t + 3 < p.nsamp) {
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
                acc[j][i] = acc[j][i + 1] = 0u;
            }
        }
        ++nflush;
    };

    // Warps synchronise through split-phase barriers, not a block barrier: ready[b] completes when all 16
    // warps have written their part of partial-sum buffer b, freeb[b] when all have consumed it; with three
    // buffers a warp only waits if another one is more than a whole group behind.
    mbar_wait(&full[0], 0);
    pre(0, 0);
    __syncwarp();
    if (lane == 0) mbar_arrive(&ready[0]);

    // st: stage of group g; sn / phn: stage and phase parity of group g + 1
    int st = 0, sn = 1 % kXStages, phn = kXStages == 1 ? 1 : 0;
    // blocks of kFlushGroups groups, one flush after each (a single flush site keeps its tail-tile
    // predicates out of the inner loop)
#pragma unroll 1
    for (int g0 = 0; g0 < ng; g0 += kFlushGroups) {
        const int g1 = min(ng, g0 + kFlushGroups);
#pragma unroll 1
        for (int g = g0; g < g1; ++g) {
            const int b = g % kPB, bn = (g + 1) % kPB;
            if (g + 1 < ng) {
                mbar_wait(&full[sn], phn);
                // buffer bn was last read by step 3 of group g + 1 - kPB: done everywhere?
                if (g + 1 >= kPB) mbar_wait(&freeb[bn], ((g + 1 - kPB) / kPB) & 1);
                pre(sn, bn);
                __syncwarp();
                if (lane == 0) mbar_arrive(&ready[bn]);
            }
            // Step 3: one word per trial, sample pair and group
            // (16-bit offsets, two per int: one 8- or 16-byte read per warp)
            int tro[KW];
            {
                uint32_t tw[KW / 2];
                const int32_t* tp = Ds + st * p.desc_ints + kDTrial + warp * (KW / 2);
                if (KW == 8) {
                    const uint4 tr = *reinterpret_cast<const uint4*>(tp);
                    tw[0] = tr.x; tw[1] = tr.y; tw[KW / 2 - 2] = tr.z; tw[KW / 2 - 1] = tr.w;
                } else {
                    const uint2 tr = *reinterpret_cast<const uint2*>(tp);
                    tw[0] = tr.x; tw[1] = tr.y;
                }
#pragma unroll
                for (int q = 0; q < KW / 2; ++q) {
                    tro[2 * q] = (int)(tw[q] & 0xffffu);
                    tro[2 * q + 1] = (int)(tw[q] >> 16);
                }
            }
            const uint32_t* ps = Ps + b * p.psw + lane;
            mbar_wait(&ready[b], (g / kPB) & 1);         // step 2 of g is done everywhere
#pragma unroll
            for (int j = 0; j < KW; ++j) {
                const uint32_t* r = ps + tro[j];
#pragma unroll
                for (int i = 0; i < NK; ++i) acc[j][i] += r[32 * i];
            }
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&freeb[b]);
                mbar_arrive(&empty[st]);                 // stage st (vectors and descriptor) may be refilled
            }
            st = sn;
            if (++sn == kXStages) { sn = 0; phn ^= 1; }
        }
        flush();
    }
}

}  // namespace

typedef void (*PsU8Kernel)(const PsU8Params, const CUtensorMap);
static PsU8Kernel psu8_kernel_for(int kw) { return kw == 8 ? dd_ps_u8_kernel<8> : dd_ps_u8_kernel<4>; }

// Descriptors for tiles of 16 kw trials; leaves p->psu8 null or not ok when the shape does not fit.
static int try_build_psu8(dd_plan* p, int kw)
{
    const int kKB = kw * kWarps, kNK = kAccPerLane / kw, kTB = 2 * 32 * kNK, kDChunk = kDTrial + kKB;
    const HostTable& h = p->host;
    const int nch = p->nchans, ndm = p->ndm;
    const int ntiles = (ndm + kKB - 1) / kKB, ngroups = (nch + kG - 1) / kG;
    // staged bytes per row: from the 16-byte aligned start of the group's first channel at the tile's
    // first trial to the end of the window of its last channel at the tile's last trial
    int64_t xwb = 0;
    for (int tile = 0; tile < ntiles; ++tile) {
        const int dfirst = tile * kKB, dlast = std::min(tile * kKB + kKB, ndm) - 1;
        for (int g = 0; g < ngroups; ++g) {
            const int c0 = g * kG, c1 = std::min(c0 + kG, nch) - 1;
            const int64_t b = h.shift[(size_t)dfirst * nch + c0] & ~15;
            xwb = std::max<int64_t>(xwb, h.shift[(size_t)dlast * nch + c1] + kTB - b);
        }
    }
    xwb = (xwb + 15) / 16 * 16;
    if (xwb > 2048) {                                     // wider than a tensor-copy box (256 x 8 bytes)
        p->ps_why = "a trial tile's input window is wider than 2048 samples (per-trial delay steps too coarse)";
        return DD_OK;
    }
    // a warp step of step 2 may read up to 2 * kChunk + 128 bytes past a row's window
    const int64_t xstage = (kG * 4 * xwb + 4 * kChunk + 384 + 127) / 128 * 128;

    // words of one parity copy of a pattern row: the largest offset of a trial in it, halved, plus
    // the kTB / 2 words every trial reads, in whole warp steps
    // warp steps of a pattern row: step c writes even-u words [62 c, 62 c + 64) and odd-u words [62 c, 62 c + 62)
    auto row_steps = [kTB](const PsRow& r) { return ((r.umax - r.umin) / 2 + kTB / 2 + kStepW - 1) / kStepW; };
    const int workers = ps_workers(ntiles);
    std::vector<int64_t> wpsw(workers, 0), wsteps(workers, 0);
    ps_parallel_tiles(ntiles, workers, [&](int tb, int te, int wk) {
        std::vector<PsRow> rows;
        int slot[kKBMax];
        for (int tile = tb; tile < te; ++tile)
            for (int g = 0; g < ngroups; ++g) {
                ps_classify(h, kG, kKB, tile, g, rows, slot);
                int64_t w = 0, n = 0;
                for (const PsRow& r : rows) {
                    n += row_steps(r);
                    w += 2 * (kStepW * row_steps(r) + 2);
                }
                wpsw[wk] = std::max(wpsw[wk], w);
                wsteps[wk] = std::max(wsteps[wk], n);
            }
    });
    int64_t psw = 0, max_steps = 0;
    for (int wk = 0; wk < workers; ++wk) {
        psw = std::max(psw, wpsw[wk]);
        max_steps = std::max(max_steps, wsteps[wk]);
    }
    const int desc_ints = kDChunk + kCE * (int)max_steps;
    const size_t smem = (size_t)kXStages * xstage + (size_t)kPB * psw * 4 +
                        (size_t)kXStages * desc_ints * 4 + (2 * kXStages + 2 * kPB) * 8;
    if (smem > (size_t)kMaxSmem) {                        // too many patterns for shared memory
        p->ps_why = "the delay patterns of a trial tile do not fit shared memory (per-trial delay steps too coarse)";
        return DD_OK;
    }

    dd_psu8_plan* t = new (std::nothrow) dd_psu8_plan;
    if (!t) return fail(DD_ERR_NOMEM, "ps u8 plan allocation failed");
    p->psu8 = t;
    t->kw = kw;
    t->ntiles = ntiles;
    t->ngroups = ngroups;
    t->desc_ints = desc_ints;
    t->xwb = (int)xwb;
    t->xstage = (int)xstage;
    t->psw = (int)psw;
    t->smem = smem;

    std::vector<int32_t> desc;
    try {
        desc.assign((size_t)ntiles * ngroups * desc_ints, 0);
    } catch (const std::bad_alloc&) {
        destroy_psu8_plan(p);
        return fail(DD_ERR_NOMEM, "ps u8 descriptor allocation failed");
    }
    const int zero_pad = kG * 4 * t->xwb;                 // byte offset of the stage's zero words
    bool bounds_ok = true;                                // every shared-memory offset written below is in range
    std::vector<char> wok(workers, 1);
    ps_parallel_tiles(ntiles, workers, [&](int tb, int te, int wk) {
    std::vector<PsRow> rows;
    int slot[kKBMax];
    std::vector<int> rowbase;
    bool bounds_ok = true;
    for (int tile = tb; tile < te; ++tile)
        for (int g = 0; g < ngroups; ++g) {
            ps_classify(h, kG, kKB, tile, g, rows, slot);
            int32_t* ds = &desc[((size_t)tile * ngroups + g) * desc_ints];
            const int c0 = g * kG, nk = std::min(kG, nch - c0);
            const int dfirst = tile * kKB, dlast = std::min(tile * kKB + kKB, ndm) - 1;
            const int base = h.shift[(size_t)dfirst * nch + c0] & ~15;   // channel c0 has the smallest delay
            ds[kDBase] = base;
            (void)dlast;
            int flat = 0, step = 0;                       // words, warp steps
            rowbase.assign(2 * rows.size(), 0);
            for (size_t r = 0; r < rows.size(); ++r) {
                const int ns = row_steps(rows[r]);
                rowbase[2 * r] = flat;                                // even-u words: (P[umin + 2 w], P[umin + 2 w + 1])
                rowbase[2 * r + 1] = flat + kStepW * ns + 2;          // odd-u words:  (P[umin + 2 w + 1], P[umin + 2 w + 2])
                // step c: lane l reads, per channel k, the aligned word with samples
                // x_k[u0 + r_k + 4 l ..+3], u0 = umin + 124 c, i.e. byte a0 + 4 l of the staged rows,
                // a0 = u0 + r_k - base: copy (a0 & 3), word (a0 >> 2) + l
                for (int c = 0; c < ns; ++c, ++step) {
                    uint16_t* ce16 = reinterpret_cast<uint16_t*>(ds + kDChunk + kCE * step);
                    int ce[6];
                    for (int k = 0; k < kG; ++k) {
                        const int rk = k == 0 ? 0 : rows[r].key[k - 1];
                        const int a0 = rows[r].umin + 2 * kStepW * c + rk - base;
                        ce[k] = k < nk ? (4 * k + (a0 & 3)) * t->xwb + (a0 & ~3) : zero_pad;
                        // every lane's read (4 bytes at ce[k] + 4 l) stays inside the stage
                        bounds_ok = bounds_ok && a0 >= 0 && ce[k] + 128 <= t->xstage;
                    }
                    ce[4] = rowbase[2 * r] + kStepW * c;
                    ce[5] = rowbase[2 * r + 1] + kStepW * c;
                    bounds_ok = bounds_ok && ce[4] + kChunk <= t->psw && ce[5] + kStepW <= t->psw;
                    for (int k = 0; k < 6; ++k) {
                        bounds_ok = bounds_ok && ce[k] >= 0 && ce[k] < 65536;
                        ce16[k] = (uint16_t)ce[k];
                    }
                }
                flat += 2 * (kStepW * ns + 2);
            }
            ds[kDNChunks] = step;
            ds[kDBytes] = 4 * (kDChunk + kCE * step);
            for (int j = 0; j < kKB; ++j) {
                const int d = std::min(tile * kKB + j, ndm - 1);
                const int o = h.shift[(size_t)d * nch + c0] - rows[slot[j]].umin;
                const int off = rowbase[2 * slot[j] + (o & 1)] + (o >> 1);
                reinterpret_cast<uint16_t*>(ds + kDTrial)[j] = (uint16_t)off;
                bounds_ok = bounds_ok && o >= 0 && off >= 0 && off < 65536 && off + kTB / 2 <= t->psw;
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
        destroy_psu8_plan(p);
        return fail(DD_ERR_NOMEM, std::string("ps u8 descriptor table: ") + cudaGetErrorString(e));
    }
    e = cudaMemcpy(t->d_desc, desc.data(), desc.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        destroy_psu8_plan(p);
        return fail(DD_ERR_CUDA, std::string("ps u8 descriptor upload: ") + cudaGetErrorString(e));
    }
    t->ok = true;
    return DD_OK;
}

int build_psu8_plan(dd_plan* p)
{
    p->psu8 = nullptr;
    if (p->ndm == 0 || p->dtype != DD_U8) return DD_OK;
    // 128-trial tiles share the pattern rows between more trials (config 2: 4.82 vs 5.01 ms); plans of
    // at most 64 trials, or whose rows do not fit then, take 64-trial tiles
    for (int kw : {8, 4}) {
        if (kw == 8 && p->ndm <= 64) continue;
        int rc = try_build_psu8(p, kw);
        if (rc != DD_OK) return rc;
        if (psu8_plan_usable(p)) break;
        destroy_psu8_plan(p);
    }
    return DD_OK;
}

void destroy_psu8_plan(dd_plan* p)
{
    if (!p->psu8) return;
    if (p->psu8->d_desc) cudaFree(p->psu8->d_desc);
    delete p->psu8;
    p->psu8 = nullptr;
}

bool psu8_plan_usable(const dd_plan* p) { return p->psu8 && p->psu8->ok; }

std::string psu8_describe(const dd_plan* p)
{
    const dd_psu8_plan* t = p->psu8;
    return "partial-sum kernel dd_ps_u8_kernel<KW=" + std::to_string(t->kw) + ">: " + std::to_string(16 * t->kw) +
           " trials x " + std::to_string(2 * 32 * kAccPerLane / t->kw) + " samples per block, " +
           std::to_string(t->smem) + " B shared memory, byte-shift front end";
}

bool psu8_args_ok(const dd_plan* p, const ExecArgs& a)
{
    if (!psu8_plan_usable(p)) return false;
    const int kTB = 2 * 32 * kAccPerLane / p->psu8->kw;
    if ((a.nsamp_out + kTB - 1) / kTB > 65535 || a.nbeams > 65535) return false;
    if ((int64_t)a.nbeams * p->nchans * 4 > 2147483647LL) return false;      // tensor-map rows / grid.x of the front end
    if ((a.nsamp_out + p->host.maxshift + 4096) / 8 >= ((int64_t)1 << 31)) return false;   // tensor coordinates
    return true;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled()
{
    static EncodeTiledFn fn = [] {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &qr) != cudaSuccess ||
            qr != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            f = nullptr;
        }
        return (EncodeTiledFn)f;
    }();
    return fn;
}

int launch_psu8(const dd_plan* p, const ExecArgs& a)
{
    const dd_psu8_plan* t = p->psu8;
    cudaStream_t st = (cudaStream_t)a.stream;
    EncodeTiledFn enc = encode_tiled();
    if (!enc) return fail(DD_ERR_CUDA, "cuTensorMapEncodeTiled is not available from this driver");
    uint8_t* W = nullptr;
    int64_t wcopy = 0, wpitch = 0;
    int rc = make_shift_copies_u8(p, a, &W, &wcopy, &wpitch);
    if (rc != DD_OK) return rc;
    // the workspace as a 2-D tensor of 8-byte elements: rows = (beam, channel, copy), wcopy bytes apart
    CUtensorMap tmap;
    const cuuint64_t dims[2] = {(cuuint64_t)(wcopy / 8), (cuuint64_t)a.nbeams * p->nchans * 4};
    const cuuint64_t strides[1] = {(cuuint64_t)wcopy};
    const cuuint32_t box[2] = {(cuuint32_t)(t->xwb / 8), 4 * kG};
    const cuuint32_t estr[2] = {1, 1};
    CUresult cr = enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT64, 2, W, dims, strides, box, estr,
                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) {
        cudaFreeAsync(W, st);
        return fail(DD_ERR_CUDA, "cuTensorMapEncodeTiled failed (" + std::to_string((int)cr) + ")");
    }
    PsU8Params q;
    q.D = (int32_t*)a.D;
    q.desc = t->d_desc;
    q.order = a.d_order;
    q.nchans = p->nchans;
    q.ndm = p->ndm;
    q.ngroups = t->ngroups;
    q.desc_ints = t->desc_ints;
    q.xwb = t->xwb;
    q.xstage = t->xstage;
    q.psw = t->psw;
    q.nsamp = a.nsamp_out;
    q.out_stride = a.out_stride;
    q.out_beam_stride = a.out_beam_stride;
    q.vec_ok = !(((uintptr_t)a.D & 15) || (a.out_stride & 3) || (a.nbeams > 1 && (a.out_beam_stride & 3)));
    const int kTB = 2 * 32 * kAccPerLane / t->kw;
    dim3 grid((unsigned)t->ntiles, (unsigned)((a.nsamp_out + kTB - 1) / kTB), (unsigned)a.nbeams);
    rc = ensure_dyn_smem((const void*)psu8_kernel_for(t->kw), t->smem);
    if (rc != DD_OK) {
        cudaFreeAsync(W, st);
        return rc;
    }
    psu8_kernel_for(t->kw)<<<grid, kThreads + 32, t->smem, st>>>(q, tmap);
    cudaError_t e = cudaGetLastError();
    cudaFreeAsync(W, st);
    if (e != cudaSuccess) return fail(DD_ERR_CUDA, std::string("ps u8 launch: ") + cudaGetErrorString(e));
    return DD_OK;
}

}  // namespace dd
