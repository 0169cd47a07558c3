// Host-side pattern classification shared by the partial-sum kernels (ps_f32.cu, ps_u8.cu).
// Not part of the C ABI; not shared with oracle/.
#pragma once

#include <algorithm>
#include <thread>
#include <vector>

#include "dd_internal.h"

namespace dd {

constexpr int kPsGMax = 8;    // largest channel group

// One pattern of relative delays r_k = s(d,c0+k) - s(d,c0), k = 1..G-1, and the range of s(d,c0)
// over the trials of the tile that have it.
struct PsRow {
    int key[kPsGMax - 1];
    int umin, umax;
};

// The distinct patterns of channel group g (G channels) among the kb sorted trials of `tile`, in
// order of first appearance; slot[j] = pattern of the tile's j-th trial (trials past the end of
// the table repeat the last one).
inline void ps_classify(const HostTable& h, int G, int kb, int tile, int g, std::vector<PsRow>& rows, int* slot)
{
    rows.clear();
    const int nch = h.nchans, ndm = h.ndm;
    const int c0 = g * G, nk = std::min(G, nch - c0);
    for (int j = 0; j < kb; ++j) {
        const int d = std::min(tile * kb + j, ndm - 1);
        const int32_t* s = &h.shift[(size_t)d * nch + c0];
        int key[kPsGMax - 1] = {0, 0, 0, 0, 0, 0, 0};
        for (int k = 1; k < nk; ++k) key[k - 1] = s[k] - s[0];
        int r = 0;
        for (; r < (int)rows.size(); ++r) {
            bool same = true;
            for (int k = 0; k < kPsGMax - 1; ++k) same = same && rows[r].key[k] == key[k];
            if (same) break;
        }
        if (r == (int)rows.size()) {
            PsRow nr;
            for (int k = 0; k < kPsGMax - 1; ++k) nr.key[k] = key[k];
            nr.umin = nr.umax = s[0];
            rows.push_back(nr);
        }
        rows[r].umin = std::min(rows[r].umin, s[0]);
        rows[r].umax = std::max(rows[r].umax, s[0]);
        slot[j] = r;
    }
}

// Runs fn(tile_begin, tile_end, worker) over [0, ntiles) on up to 16 host threads (the descriptor
// passes are independent per trial tile; config 3 has 64 tiles x 512 groups x 64 trials).
inline int ps_workers(int ntiles)
{
    const unsigned hw = std::thread::hardware_concurrency();
    return std::max(1, std::min({ntiles, (int)(hw ? hw : 1), 16}));
}
template <typename F>
inline void ps_parallel_tiles(int ntiles, int workers, F fn)
{
    if (workers <= 1) {
        fn(0, ntiles, 0);
        return;
    }
    std::vector<std::thread> th;
    const int per = (ntiles + workers - 1) / workers;
    for (int w = 0; w < workers; ++w) {
        const int b = std::min(ntiles, w * per), e = std::min(ntiles, b + per);
        th.emplace_back([=] { fn(b, e, w); });
    }
    for (auto& t : th) t.join();
}

}  // namespace dd
