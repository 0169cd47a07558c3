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
//      memory.  All rows of a tile sit on one grid of 32-word chunks of u.  A warp takes a "segment":
//      a run of up to 8 patterns that need the same chunk and in which every r_k takes at most two
//      adjacent values a_k, a_k + 1 (adjacent trials move a relative delay by less than a sample).  It
//      loads both candidates x_k[u + a_k], x_k[u + a_k + 1] of every channel into REGISTERS once
//      (2 G - 1 shared-memory loads per lane) and forms the row words of all patterns of the run from
//      them: per pattern G - 1 selects (predicates from one R2P), G - 1 adds and one store, no
//      further load -- against G loads per row word when every row is formed on its own;
//   3. adds, for every trial d and sample t of the tile, ONE word:  acc += P_{pattern(d)}[t + s(d,c0)].
// Step 3 costs one shared-memory word per FOUR channel-adds; step 2 one store per row word plus
// (2 G + 7) / 32 loads per segment word.  Descriptors (windows, segments, per-trial row offsets) are built on
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
constexpr int kXStages = 3;               // staged groups in flight
constexpr int kPB = 3;                    // partial-sum buffers: step 2 may run two groups ahead of step 3
constexpr int kMaxSmem = 224 * 1024;

// descriptor layout (ints), one per (trial tile, channel group)
constexpr int kCW = 32;                   // words of a chunk: one u per lane
constexpr int kPad = 64;                  // spare words behind the staged vectors (chunk-aligned rows read past them)
constexpr int kDNSegs = 0;                // number of segments (work items of step 2)
constexpr int kDBytes = 1;                // bytes of this descriptor that are in use (multiple of 16)
constexpr int kDEnt = 2;                  // first int of the segment blocks
constexpr int kDBase = 4;                 // [8]  first staged word of channel k, relative to t0 (multiple of 4)
constexpr int kDLen = 12;                 // [8]  words to stage (multiple of 4; 0 for a missing channel)
constexpr int kDTrial = 20;               // [KB] flat word offset of trial j's first operand in the partial sums
// kDTrial + KB:                             [12] uint16 x 17: warp w takes segments wstart[w] .. wstart[w+1]-1
// kDTrial + KB + 12 (= kDEnt):              [nsegs][8] segment blocks.  A segment is a run of at most kNP patterns that
//                                                need the same chunk and in which every r_k takes at most two values,
//                                                a_k and a_k + 1:
//                   [4] uint16 x 8: word offset, from the stage's first word, of lane 0's operand x_k[u + a_k]
//                                   (a missing channel, and k >= G, points at the zero pad)
//                   [4] uint16 x 8: one entry per pattern: bit k-1 = (r_k == a_k + 1), k = 1..G-1; bits 7-15 = 1 + word
//                                   offset / 32 of the pattern's 32 row words in the partial-sum buffer; 0 = no pattern
constexpr int kDWarpInts = 12;
constexpr int kNP = 8;                    // patterns per segment
constexpr int kSegInts = 8;

struct PsParams {
    const float* X;
    float* D;
    const int32_t* desc;
    const int32_t* order;
    int nchans, ndm, ngroups, desc_ints, xw, psw;
    int64_t nsamp, row_valid;      // row_valid: words of a channel row that may be read (multiple of 4)
    int64_t in_stride, in_beam_stride, out_stride, out_beam_stride;
};

// One row word of a pattern: ((x0 + x1) + x2) + ... with x_k = b[k] where bit k-1 of the pattern's entry e is set
// (r_k = a_k + 1), else a[k].  The association depends on nothing but G.
template <int G> __device__ __forceinline__ float pattern_sum(const float (&a)[G], const float (&b)[G], uint32_t e)
{
    float s = a[0];
#pragma unroll
    for (int k = 1; k < G; ++k) s += (e >> (k - 1)) & 1u ? b[k] : a[k];
    return s;
}

template <int G, int KW>
__global__ void __launch_bounds__(kThreads + 32, 1)
dd_ps_f32_kernel(const PsParams p)
{
    constexpr int NK = kAccPerLane / KW, KB = KW * kWarps, TB = 32 * NK;
    extern __shared__ __align__(128) uint8_t smem_raw[];
    const int xstage = G * p.xw + kPad;                                        // words; the last kPad stay zero
    float* Xs = reinterpret_cast<float*>(smem_raw);                            // [kXStages][xstage]
    float* Ps = Xs + kXStages * xstage;                                        // [2][psw]
    int32_t* Ds = reinterpret_cast<int32_t*>(Ps + kPB * p.psw);                  // [kXStages][desc_ints]
    uint64_t* full = reinterpret_cast<uint64_t*>(Ds + kXStages * p.desc_ints); // [kXStages]
    uint64_t* empty = full + kXStages;                                         // [kXStages]
    uint64_t* ready = empty + kXStages;                                        // [2] partial sums complete
    uint64_t* freeb = ready + kPB;                                               // [2] partial sums consumed

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
        for (int b = 0; b < kPB; ++b) {
            mbar_init(&ready[b], kWarps);
            mbar_init(&freeb[b], kWarps);
        }
        mbar_fence_init();
    }
    if (threadIdx.x < kXStages * kPad)
        Xs[(threadIdx.x / kPad) * xstage + G * p.xw + (threadIdx.x % kPad)] = 0.0f;
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
    // Step 2: the pattern rows of group g into partial-sum buffer `buf`.  The rows sit on a common grid of
    // chunks of 32 consecutive u (one per lane).  A segment is a run of patterns that need the same chunk and
    // whose relative delays take at most two adjacent values per channel: the warp loads both candidates
    // x_k[u + a_k], x_k[u + a_k + 1] of every channel into registers ONCE (2 G - 1 loads) and then forms the
    // row words of every pattern of the run from registers -- per pattern and word G - 1 selects, G - 1 adds
    // and one store, no further shared-memory read.  The host split the segments evenly over the 16 warps.
    auto pre = [&](int st, int buf) {
        const int32_t* ds = Ds + st * p.desc_ints;
        const uint32_t xa = smem_u32(Xs + st * xstage) + lane * 4;
        const uint32_t pa = smem_u32(Ps + buf * p.psw) + lane * 4 - kCW * 4;    // entries hold 1 + chunk index
        const uint16_t* ws = reinterpret_cast<const uint16_t*>(ds + kDTrial + KB);
        const uint4* blk = reinterpret_cast<const uint4*>(ds + kDTrial + KB + kDWarpInts);
        const int cend = ws[warp + 1];
        for (int c = ws[warp]; c < cend; ++c) {
            const uint4 o = blk[2 * c], en = blk[2 * c + 1];
            const uint32_t ow[4] = {o.x, o.y, o.z, o.w}, ew[4] = {en.x, en.y, en.z, en.w};
            float a[G], b[G];
#pragma unroll
            for (int k = 0; k < G; ++k) {
                const uint32_t ad = xa + ((ow[k >> 1] >> (16 * (k & 1))) & 0xffffu) * 4;
                a[k] = lds_f32(ad);
                b[k] = k ? lds_f32(ad + 4) : 0.0f;
            }
#pragma unroll
            for (int i = 0; i < kNP; ++i) {
                const uint32_t e = ew[i >> 1] >> (16 * (i & 1));               // entry of the run's i-th pattern
                if (!(e & 0xff80u)) break;
                sts_f32(pa + (e & 0xff80u), pattern_sum<G>(a, b, e));
            }
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
        const int b = g % kPB, bn = (g + 1) % kPB;
        if (g + 1 < ng) {
            mbar_wait(&full[sn], phn);
            // buffer bn was last read by step 3 of group g + 1 - kPB: done everywhere?
            if (g + 1 >= kPB) mbar_wait(&freeb[bn], ((g + 1 - kPB) / kPB) & 1);
            pre(sn, bn);
            __syncwarp();
            if (lane == 0) mbar_arrive(&ready[bn]);
        }
        // Step 3: one word per trial, sample and group
        int tro[KW];
#pragma unroll
        for (int q = 0; q < KW / 4; ++q) {
            const int4 tr = *reinterpret_cast<const int4*>(Ds + st * p.desc_ints + kDTrial + warp * KW + 4 * q);
            tro[4 * q] = tr.x; tro[4 * q + 1] = tr.y; tro[4 * q + 2] = tr.z; tro[4 * q + 3] = tr.w;
        }
        const float* ps = Ps + b * p.psw + lane;
        mbar_wait(&ready[b], (g / kPB) & 1);                                // step 2 of g is done everywhere
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

// Placement of the pattern rows of one (tile, group) on the common grid of kCW-word chunks, and the work
// list of step 2.  Chunk c covers u0 + kCW c .. + kCW - 1 with u0 the smallest s(d, c0) of the tile; row r
// occupies chunks cb[r] .. ce[r] and sits at word rowbase[r] of the partial-sum buffer.  Items = (chunk,
// row) pairs in chunk-major order, rows in order of first appearance; a segment is a run of items of one
// chunk; warp w takes segments wstart[w] .. wstart[w+1]-1, cut so that every warp gets about the same cost.
// Orders the patterns of a (tile, group) so that neighbours differ in few r_k: by the sum of the relative
// delays, then lexicographically.  (Where the r_k only jitter between two adjacent integers with the
// fractional part of s(d, c0), the patterns form a chain along which one r_k changes at a time; where they
// grow with the trial, this is the order of first appearance.)  slot[] is renumbered accordingly.
void ps_chain_order(std::vector<PsRow>& rows, int* slot, int kb)
{
    const int nr = (int)rows.size();
    std::vector<int> idx(nr), inv(nr);
    for (int r = 0; r < nr; ++r) idx[r] = r;
    auto weight = [&](int r) { int w = 0; for (int k = 0; k < kPsGMax - 1; ++k) w += rows[r].key[k]; return w; };
    std::sort(idx.begin(), idx.end(), [&](int a, int b) {
        const int wa = weight(a), wb = weight(b);
        if (wa != wb) return wa < wb;
        for (int k = 0; k < kPsGMax - 1; ++k)
            if (rows[a].key[k] != rows[b].key[k]) return rows[a].key[k] < rows[b].key[k];
        return a < b;
    });
    std::vector<PsRow> out(nr);
    for (int r = 0; r < nr; ++r) { out[r] = rows[idx[r]]; inv[idx[r]] = r; }
    rows.swap(out);
    for (int j = 0; j < kb; ++j) slot[j] = inv[slot[j]];
}

struct PsSeg { int chunk, first, count; int a[kPsGMax - 1]; };
struct PsLayout {
    int u0 = 0, flat = 0, npw = 0;
    std::vector<int> cb, ce, rowbase, item_chunk, item_row;
    std::vector<PsSeg> segs;
    int wstart[kWarps + 1];
};

void ps_layout(const std::vector<PsRow>& rows, int G, int kTB, PsLayout& L)
{
    const int nr = (int)rows.size();
    L.cb.assign(nr, 0);
    L.ce.assign(nr, 0);
    L.rowbase.assign(nr, 0);
    L.u0 = rows[0].umin;
    for (const PsRow& r : rows) L.u0 = std::min(L.u0, r.umin);
    L.flat = 0;
    int nch = 0;
    for (int r = 0; r < nr; ++r) {
        L.cb[r] = (rows[r].umin - L.u0) / kCW;
        L.ce[r] = (rows[r].umax + kTB - 1 - L.u0) / kCW;
        L.rowbase[r] = L.flat;
        L.flat += kCW * (L.ce[r] - L.cb[r] + 1);
        nch = std::max(nch, L.ce[r] + 1);
    }
    L.item_chunk.clear();
    L.item_row.clear();
    for (int c = 0; c < nch; ++c)
        for (int r = 0; r < nr; ++r)
            if (c >= L.cb[r] && c <= L.ce[r]) {
                L.item_chunk.push_back(c);
                L.item_row.push_back(r);
            }
    // segments: greedy runs; a run ends at a new chunk, at kNP patterns, when some r_k would span more than two
    // adjacent values, and where the cost so far says the next warp should start (loading a run's operands
    // costs about as much as three pattern words)
    const int header = 3;
    const int ni = (int)L.item_row.size();
    L.npw = ni;
    L.segs.clear();
    int lo[kPsGMax - 1], hi[kPsGMax - 1];
    auto fits_run = [&](int r) {
        for (int k = 0; k < G - 1; ++k)
            if (std::max(hi[k], rows[r].key[k]) - std::min(lo[k], rows[r].key[k]) > 1) return false;
        return true;
    };
    // first pass: runs without balancing, to know the total cost
    int total = 0;
    {
        int cnt = 0;
        for (int i = 0; i < ni; ++i) {
            const int r = L.item_row[i];
            const bool start = i == 0 || L.item_chunk[i] != L.item_chunk[i - 1] || cnt == kNP || !fits_run(r);
            if (start) {
                total += header;
                cnt = 0;
                for (int k = 0; k < G - 1; ++k) lo[k] = hi[k] = rows[r].key[k];
            }
            for (int k = 0; k < G - 1; ++k) {
                lo[k] = std::min(lo[k], rows[r].key[k]);
                hi[k] = std::max(hi[k], rows[r].key[k]);
            }
            ++cnt;
            ++total;
        }
    }
    int w = 0, acc = 0;
    L.wstart[0] = 0;
    for (int i = 0; i < ni; ++i) {
        const int r = L.item_row[i];
        bool start = i == 0 || L.item_chunk[i] != L.item_chunk[i - 1] || L.segs.back().count == kNP || !fits_run(r);
        if (start) acc += header;                        // (the operands reloaded after a balancing cut are not counted)
        if (i > 0 && w < kWarps - 1 && (int64_t)acc * kWarps >= (int64_t)total * (w + 1)) {
            L.wstart[++w] = (int)L.segs.size();
            start = true;
        }
        if (start) {
            PsSeg sg;
            sg.chunk = L.item_chunk[i];
            sg.first = i;
            sg.count = 0;
            for (int k = 0; k < kPsGMax - 1; ++k) sg.a[k] = 0;
            L.segs.push_back(sg);
            for (int k = 0; k < G - 1; ++k) lo[k] = hi[k] = rows[r].key[k];
        }
        for (int k = 0; k < G - 1; ++k) {
            lo[k] = std::min(lo[k], rows[r].key[k]);
            hi[k] = std::max(hi[k], rows[r].key[k]);
            L.segs.back().a[k] = lo[k];
        }
        ++L.segs.back().count;
        ++acc;
    }
    while (w < kWarps) L.wstart[++w] = (int)L.segs.size();
}

// Shared-memory need and modelled cost per output tile for group size G and tile shape kw.  Shared-memory
// wavefronts: step 3 takes KB * NK + KB per group (one word per trial and sample, the row offsets), step 2
// 2 G + 9 per segment (two 16-byte block reads, the operands) and one store per pattern word.  Issue slots:
// step 3 about 2.8 per word, a segment about 30 + 4 G, a pattern word about 5 + 3 (G - 1) instructions; four
// schedulers.  The cost is the larger of the two.
PsShape shape_for(const HostTable& h, int G, int kw)
{
    PsShape o;
    const int kKB = kw * kWarps, kNK = kAccPerLane / kw, kTB = 32 * kNK, kDChunk = kDTrial + kKB;
    const int ntiles = (h.ndm + kKB - 1) / kKB, ngroups = (h.nchans + G - 1) / G;
    const int64_t spread = max_tile_spread(h, kKB);
    o.xw = (kTB + spread + 3 + 3) / 4 * 4 + kPad;
    const int workers = ps_workers(ntiles);
    std::vector<int64_t> wpsw(workers, 0), wsegs(workers, 0), wpw(workers, 0), wmax(workers, 0);
    ps_parallel_tiles(ntiles, workers, [&](int tb, int te, int wk) {
        std::vector<PsRow> rows;
        PsLayout L;
        int slot[kKBMax];
        for (int tile = tb; tile < te; ++tile)
            for (int g = 0; g < ngroups; ++g) {
                ps_classify(h, G, kKB, tile, g, rows, slot);
                ps_chain_order(rows, slot, kKB);
                ps_layout(rows, G, kTB, L);
                wpsw[wk] = std::max<int64_t>(wpsw[wk], L.flat);
                wmax[wk] = std::max<int64_t>(wmax[wk], (int64_t)L.segs.size());
                wsegs[wk] += (int64_t)L.segs.size();
                wpw[wk] += L.npw;
            }
    });
    int64_t segs = 0, pw = 0, maxsegs = 0;
    for (int wk = 0; wk < workers; ++wk) {
        o.psw = std::max(o.psw, wpsw[wk]);
        maxsegs = std::max(maxsegs, wmax[wk]);
        segs += wsegs[wk];
        pw += wpw[wk];
    }
    o.desc_ints = (int)(kDChunk + kDWarpInts + kSegInts * maxsegs + 4);
    o.smem = (size_t)kXStages * (G * o.xw + kPad) * 4 + (size_t)kPB * o.psw * 4 +
             (size_t)kXStages * o.desc_ints * 4 + (2 * kXStages + 2 * kPB) * 8;
    o.fits = G * o.xw + kPad < 65536 && o.psw / kCW <= 511 && maxsegs < 65536 && o.smem <= (size_t)kMaxSmem;
    const double tg = (double)ntiles * ngroups;
    const double lsu = tg * (kKB * kNK + kKB) + (double)segs * (2 * G + 9) + (double)pw;
    const double issue = (tg * 2.8 * kKB * kNK + (30.0 + 4.0 * G) * segs + (5.0 + 3.0 * (G - 1)) * pw) / 4.0;
    o.cost = std::max(lsu / 0.85, issue / 0.8);
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
    const int zero_pad = G * t->xw;                       // word offset of the stage's kPad zero words
    bool bounds_ok = true;                                // every shared-memory offset written below is in range
    const int workers = ps_workers(ntiles);
    std::vector<char> wok(workers, 1);
    ps_parallel_tiles(ntiles, workers, [&](int tb, int te, int wk) {
    std::vector<PsRow> rows;
    PsLayout L;
    int slot[kKBMax];
    bool bounds_ok = true;
    for (int tile = tb; tile < te; ++tile)
        for (int g = 0; g < ngroups; ++g) {
            ps_classify(h, G, kKB, tile, g, rows, slot);
            ps_chain_order(rows, slot, kKB);
            ps_layout(rows, G, kTB, L);
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
            // word e of row r's storage is u = u0 + kCW cb[r] + e; channel k supplies x_k[u + r_k], staged at word
            // (u + r_k - base_k) of its vector.  The first chunk of a row starts up to kCW - 1 words before the
            // row's first valid u and its last chunk ends as many after: those words read neighbouring staged
            // data (for k = 0 never below the stage: u >= u0 >= base_0) and are never used by step 3.
            const int nsegs = (int)L.segs.size();
            const int ent0 = kDChunk + kDWarpInts;
            uint16_t* ws = reinterpret_cast<uint16_t*>(ds + kDChunk);
            for (int w = 0; w <= kWarps; ++w) ws[w] = (uint16_t)L.wstart[w];
            for (int sg = 0; sg < nsegs; ++sg) {
                const PsSeg& S = L.segs[sg];
                uint16_t* o16 = reinterpret_cast<uint16_t*>(ds + ent0 + kSegInts * sg);
                uint16_t* e16 = o16 + 8;
                for (int k = 0; k < 8; ++k) {
                    const int ak = k == 0 ? 0 : (k < G ? S.a[k - 1] : 0);
                    const int off = k < nk ? k * t->xw + L.u0 + kCW * S.chunk + ak - base[k] : zero_pad;
                    // both candidates of every lane (words off + l and off + l + 1) stay inside the stage
                    bounds_ok = bounds_ok && off >= 0 && off + 1 + kCW <= G * t->xw + kPad;
                    o16[k] = (uint16_t)off;
                }
                bounds_ok = bounds_ok && S.count >= 1 && S.count <= kNP;
                for (int i = 0; i < S.count; ++i) {
                    const int r = L.item_row[S.first + i];
                    const int store = L.rowbase[r] + kCW * (S.chunk - L.cb[r]);
                    bounds_ok = bounds_ok && store >= 0 && store + kCW <= t->psw && store / kCW < 511;
                    uint32_t bits = 0;
                    for (int k = 1; k < G; ++k) {
                        const int dk = rows[r].key[k - 1] - S.a[k - 1];
                        bounds_ok = bounds_ok && (dk == 0 || dk == 1);
                        bits |= (uint32_t)(dk & 1) << (k - 1);
                    }
                    e16[i] = (uint16_t)(bits | (uint32_t)(store / kCW + 1) << 7);
                }
            }
            bounds_ok = bounds_ok && ent0 + kSegInts * nsegs + 4 <= desc_ints && nsegs < 65536;
            ds[kDNSegs] = nsegs;
            ds[kDEnt] = ent0;
            ds[kDBytes] = (4 * (ent0 + kSegInts * nsegs) + 15) / 16 * 16;
            for (int j = 0; j < kKB; ++j) {
                const int d = std::min(tile * kKB + j, ndm - 1);
                const int s0 = h.shift[(size_t)d * nch + c0];
                const int r = slot[j];
                ds[kDTrial + j] = L.rowbase[r] + (s0 - (L.u0 + kCW * L.cb[r]));
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
