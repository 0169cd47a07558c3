// The thesis' two approximate variants of direct dedispersion, float32:
//   A. time binning: trials above twice the diagonal DM run on input summed over
//      2, 4, 8, ... adjacent samples ("downfactor the time series by a factor of 2 by summing adjacent
//      samples"), at the correspondingly longer sampling time;
//   B. subband dedispersion (§2.1.3): step 1 dedisperses subbands of N'_c channels at one
//      nominal DM per N'_DM trials, step 2 dedisperses the reduced filterbank of subband series at every
//      trial's own DM.
// Both "reuse the same kernel on reduced data": every dedispersion step is a dd_plan of this library
// (partial-sum / generic / direct kernels), created once per composite object; this file adds the
// pairwise-sum kernel and the orchestration (readings R28-R33).  The adds saved are the
// method's; nothing here changes the exact path.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <new>
#include <vector>

#include "dd_internal.h"

struct dd_timebin {
    int nchans = 0, ndm = 0, nlevels = 0;
    double dm_diag = 0;
    std::vector<int32_t> level;          // per trial
    std::vector<int> first, count;       // per level: first row, number of trials
    std::vector<dd_plan*> plans;         // per level (null when the level has no trial)
};

struct dd_subband {
    int nchans = 0, ndm = 0, ncs = 0, nds = 0, nsb = 0, nnom = 0;
    int64_t ms1 = 0, ms2 = 0;
    std::vector<dd_plan*> sub;           // per subband: its channels at the nominal DMs
    std::vector<dd_plan*> grp;           // per nominal group: the reduced filterbank at the group's DMs
    // the plans of a step are independent small launches: they are spread over a few internal streams
    // (fork from / join to the caller's stream with events) so that their ramp-up and tails overlap
    static constexpr int kStreams = 4;
    cudaStream_t aux[kStreams] = {nullptr, nullptr, nullptr, nullptr};
    cudaEvent_t fork = nullptr, join[kStreams] = {nullptr, nullptr, nullptr, nullptr};
};

namespace dd {

namespace {

// Y[r][i] = X[r][2i] + X[r][2i+1]
__global__ void __launch_bounds__(256)
dd_downsample2_kernel(const float* __restrict__ X, float* __restrict__ Y, int64_t n_out, int64_t stride_in,
                      int64_t stride_out)
{
    const int64_t r = blockIdx.y;
    const float* x = X + r * stride_in;
    float* y = Y + r * stride_out;
    const bool vec = ((((uintptr_t)x) & 7) == 0);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_out; i += (int64_t)gridDim.x * blockDim.x) {
        float a, b;
        if (vec) {
            const float2 v = __ldg(reinterpret_cast<const float2*>(x) + i);
            a = v.x;
            b = v.y;
        } else {
            a = __ldg(x + 2 * i);
            b = __ldg(x + 2 * i + 1);
        }
        y[i] = a + b;
    }
}

const double kDM = 4148.808;   // eq 1.14

bool non_decreasing(const double* dm, int n)
{
    for (int i = 1; i < n; ++i)
        if (!(dm[i] >= dm[i - 1])) return false;
    return true;
}

}  // namespace

int downsample2(const float* X, float* Y, int64_t nrows, int64_t n_in, int64_t stride_in, int64_t stride_out,
                void* cuda_stream)
{
    if (nrows < 0 || n_in < 0) return fail(DD_ERR_BAD_ARG, "bad nrows / n_in");
    const int64_t n_out = n_in / 2;
    if (nrows == 0 || n_out == 0) return DD_OK;
    if (!X || !Y) return fail(DD_ERR_BAD_ARG, "X or Y is null");
    if (stride_in < n_in || stride_out < n_out) return fail(DD_ERR_BAD_ARG, "stride is shorter than the row");
    for (int64_t r0 = 0; r0 < nrows; r0 += 65535) {
        const int64_t nr = std::min<int64_t>(65535, nrows - r0);
        dim3 grid((unsigned)std::min<int64_t>((n_out + 255) / 256, 1024), (unsigned)nr);
        dd_downsample2_kernel<<<grid, 256, 0, (cudaStream_t)cuda_stream>>>(X + r0 * stride_in, Y + r0 * stride_out,
                                                                           n_out, stride_in, stride_out);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(DD_ERR_CUDA, std::string("downsample launch: ") + cudaGetErrorString(e));
    return DD_OK;
}

double diagonal_dm(int nchans, double fch1, double foff, double tsamp)
{
    if (nchans < 2 || foff == 0.0) return INFINITY;
    const double f1 = fch1 + (double)(nchans - 1) * foff, f2 = fch1 + (double)(nchans - 2) * foff;
    return tsamp / (kDM * (1.0 / (f1 * f1) - 1.0 / (f2 * f2)));
}

}  // namespace dd

using namespace dd;

extern "C" {

int dd_downsample2_f32(const float* X, float* Y, int64_t nrows, int64_t n_in, int64_t stride_in,
                       int64_t stride_out, void* cuda_stream)
{
    return downsample2(X, Y, nrows, n_in, stride_in, stride_out, cuda_stream);
}

double dd_diagonal_dm(int nchans, double fch1, double foff, double tsamp)
{
    return diagonal_dm(nchans, fch1, foff, tsamp);
}

// ------------------------------------------------------------------------------ time binning

void dd_timebin_destroy(dd_timebin* t)
{
    if (!t) return;
    for (dd_plan* p : t->plans)
        if (p) dd_plan_destroy(p);
    delete t;
}

int dd_timebin_create(dd_timebin** out, int nchans, double fch1, double foff, double tsamp, const double* dm_list,
                      int ndm, double dm_diag, int max_level)
{
    if (!out) return fail(DD_ERR_BAD_ARG, "out is null");
    *out = nullptr;
    if (max_level < 0 || max_level > 16) return fail(DD_ERR_BAD_ARG, "max_level must be 0..16");
    // argument validation of the filterbank and the DM list (same rules as dd_plan_create)
    if (host_max_shift(nchans, fch1, foff, tsamp, dm_list, ndm) < 0) return DD_ERR_BAD_ARG;
    if (!non_decreasing(dm_list, ndm)) return fail(DD_ERR_BAD_ARG, "dm_list must be non-decreasing (R30)");
    if (!(dm_diag > 0.0)) dm_diag = diagonal_dm(nchans, fch1, foff, tsamp);
    dd_timebin* t = new (std::nothrow) dd_timebin;
    if (!t) return fail(DD_ERR_NOMEM, "allocation failed");
    t->nchans = nchans;
    t->ndm = ndm;
    t->dm_diag = dm_diag;
    t->level.resize(ndm);
    int top = 0;
    for (int i = 0; i < ndm; ++i) {
        int k = 0;
        if (dm_list[i] >= 2.0 * dm_diag) k = std::min(max_level, (int)std::floor(std::log2(dm_list[i] / dm_diag)));
        t->level[i] = k;
        top = std::max(top, k);
    }
    t->nlevels = ndm ? top + 1 : 0;
    t->first.assign(t->nlevels, 0);
    t->count.assign(t->nlevels, 0);
    t->plans.assign(t->nlevels, nullptr);
    for (int i = 0; i < ndm; ++i) {
        if (t->count[t->level[i]] == 0) t->first[t->level[i]] = i;
        ++t->count[t->level[i]];
    }
    for (int k = 0; k < t->nlevels; ++k) {
        if (!t->count[k]) continue;
        int rc = dd_plan_create(&t->plans[k], DD_F32, nchans, fch1, foff, std::ldexp(tsamp, k), dm_list + t->first[k],
                                t->count[k]);
        if (rc != DD_OK) {
            dd_timebin_destroy(t);
            return rc;
        }
    }
    *out = t;
    return DD_OK;
}

int dd_timebin_levels(const dd_timebin* t, int32_t* level_of_trial)
{
    if (!t) return fail(DD_ERR_BAD_ARG, "null argument");
    if (level_of_trial)
        for (int i = 0; i < t->ndm; ++i) level_of_trial[i] = t->level[i];
    return t->nlevels;
}

int64_t dd_timebin_input_samples(const dd_timebin* t, int64_t nsamp_out)
{
    if (!t || nsamp_out < 0) return fail(DD_ERR_BAD_ARG, "bad argument");
    int64_t need = 0;
    for (int k = 0; k < t->nlevels; ++k)
        if (t->plans[k]) need = std::max(need, ((nsamp_out >> k) + dd_plan_max_shift(t->plans[k])) << k);
    return need;
}

int dd_timebin_execute(dd_timebin* t, const float* X, int64_t in_stride, int64_t n_in, float* D, int64_t out_stride,
                       int64_t nsamp_out, void* cuda_stream)
{
    if (!t) return fail(DD_ERR_BAD_ARG, "null argument");
    if (nsamp_out < 0) return fail(DD_ERR_BAD_ARG, "nsamp_out must be >= 0");
    if (t->ndm == 0 || nsamp_out == 0) return DD_OK;
    if (!X || !D) return fail(DD_ERR_BAD_ARG, "X or D is null");
    if (n_in < dd_timebin_input_samples(t, nsamp_out) || in_stride < n_in)
        return fail(DD_ERR_BAD_ARG, "input rows are shorter than dd_timebin_input_samples(nsamp_out)");
    if (out_stride < nsamp_out) return fail(DD_ERR_BAD_ARG, "out_stride is shorter than nsamp_out");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // binned copies: level k rows hold n_in >> k samples, pitch rounded to 64 elements; one workspace for all
    std::vector<int64_t> pitch(t->nlevels, 0), off(t->nlevels, 0);
    int64_t total = 0;
    for (int k = 1; k < t->nlevels; ++k) {
        pitch[k] = ((n_in >> k) + 63) / 64 * 64;
        off[k] = total;
        total += pitch[k] * t->nchans;
    }
    float* ws = nullptr;
    if (total > 0) {
        int rc = workspace_alloc((void**)&ws, (size_t)total * sizeof(float), cuda_stream);
        if (rc != DD_OK) return rc;
    }
    int rc = DD_OK;
    const float* cur = X;
    int64_t cur_stride = in_stride, cur_n = n_in;
    for (int k = 0; k < t->nlevels && rc == DD_OK; ++k) {
        if (k > 0) {
            float* nxt = ws + off[k];
            rc = downsample2(cur, nxt, t->nchans, cur_n, cur_stride, pitch[k], cuda_stream);
            cur = nxt;
            cur_stride = pitch[k];
            cur_n >>= 1;
        }
        const int64_t nout = nsamp_out >> k;
        if (rc == DD_OK && t->plans[k] && nout > 0)
            rc = dd_execute(t->plans[k], cur, cur_stride, 0, D + (int64_t)t->first[k] * out_stride, out_stride, 0, nout, 1,
                            cuda_stream);
    }
    if (ws) cudaFreeAsync(ws, st);
    return rc;
}

// ------------------------------------------------------------------------------ subband dedispersion

// The plans of the two steps have few channels and trials ("tiny": AUTO would give them the direct kernel, which
// is built for short series such as BASELINE.json configs[0]) but run over the whole observation: the partial-sum
// kernel where it takes the plan, else the shared-memory channel-vector kernel -- 1.2-1.8x faster than the direct
// kernel on 2^17 samples.  The choice is fixed per plan, so every call adds in the same order.
static void prefer_streaming_kernel(dd_plan* p)
{
    dd_plan_set_kernel(p, dd::ps_plan_usable(p) ? DD_KERNEL_PS : DD_KERNEL_GENERIC);
}

void dd_subband_destroy(dd_subband* s)
{
    if (!s) return;
    for (dd_plan* p : s->sub)
        if (p) dd_plan_destroy(p);
    for (dd_plan* p : s->grp)
        if (p) dd_plan_destroy(p);
    for (int i = 0; i < dd_subband::kStreams; ++i) {
        if (s->aux[i]) cudaStreamDestroy(s->aux[i]);
        if (s->join[i]) cudaEventDestroy(s->join[i]);
    }
    if (s->fork) cudaEventDestroy(s->fork);
    delete s;
}

int dd_subband_create(dd_subband** out, int nchans, double fch1, double foff, double tsamp, const double* dm_list,
                      int ndm, int chans_per_subband, int dms_per_nominal)
{
    if (!out) return fail(DD_ERR_BAD_ARG, "out is null");
    *out = nullptr;
    if (chans_per_subband < 1 || dms_per_nominal < 1) return fail(DD_ERR_BAD_ARG, "group sizes must be >= 1");
    if (host_max_shift(nchans, fch1, foff, tsamp, dm_list, ndm) < 0) return DD_ERR_BAD_ARG;
    if (!non_decreasing(dm_list, ndm)) return fail(DD_ERR_BAD_ARG, "dm_list must be non-decreasing (R30)");
    dd_subband* s = new (std::nothrow) dd_subband;
    if (!s) return fail(DD_ERR_NOMEM, "allocation failed");
    s->nchans = nchans;
    s->ndm = ndm;
    s->ncs = chans_per_subband;
    s->nds = dms_per_nominal;
    s->nsb = (nchans + chans_per_subband - 1) / chans_per_subband;
    s->nnom = (ndm + dms_per_nominal - 1) / dms_per_nominal;
    std::vector<double> noms(s->nnom);
    for (int g = 0; g < s->nnom; ++g) {
        const int d0 = g * dms_per_nominal, d1 = std::min(ndm, d0 + dms_per_nominal);
        noms[g] = dm_list[d0 + (d1 - d0 - 1) / 2];                      // the group's middle trial (R32)
    }
    s->sub.assign(s->nsb, nullptr);
    s->grp.assign(s->nnom, nullptr);
    int rc = DD_OK;
    for (int b = 0; b < s->nsb && rc == DD_OK && ndm > 0; ++b) {
        const int c0 = b * chans_per_subband, c1 = std::min(nchans, c0 + chans_per_subband);
        rc = dd_plan_create(&s->sub[b], DD_F32, c1 - c0, fch1 + (double)c0 * foff, foff, tsamp, noms.data(), s->nnom);
        if (rc == DD_OK) s->ms1 = std::max(s->ms1, dd_plan_max_shift(s->sub[b]));
        if (rc == DD_OK) prefer_streaming_kernel(s->sub[b]);
    }
    for (int g = 0; g < s->nnom && rc == DD_OK; ++g) {
        const int d0 = g * dms_per_nominal, d1 = std::min(ndm, d0 + dms_per_nominal);
        rc = dd_plan_create(&s->grp[g], DD_F32, s->nsb, fch1, (double)chans_per_subband * foff, tsamp, dm_list + d0,
                            d1 - d0);
        if (rc == DD_OK) s->ms2 = std::max(s->ms2, dd_plan_max_shift(s->grp[g]));
        if (rc == DD_OK) prefer_streaming_kernel(s->grp[g]);
    }
    if (rc == DD_OK && ndm > 0) {
        cudaError_t e = cudaEventCreateWithFlags(&s->fork, cudaEventDisableTiming);
        for (int i = 0; i < dd_subband::kStreams && e == cudaSuccess; ++i) {
            e = cudaStreamCreateWithFlags(&s->aux[i], cudaStreamNonBlocking);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->join[i], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) rc = fail(DD_ERR_CUDA, std::string("subband streams: ") + cudaGetErrorString(e));
    }
    if (rc != DD_OK) {
        dd_subband_destroy(s);
        return rc;
    }
    *out = s;
    return DD_OK;
}

int64_t dd_subband_max_shift(const dd_subband* s)
{
    if (!s) return fail(DD_ERR_BAD_ARG, "null argument");
    return s->ms1 + s->ms2;
}

int dd_subband_execute(dd_subband* s, const float* X, int64_t in_stride, float* D, int64_t out_stride,
                       int64_t nsamp_out, void* cuda_stream)
{
    if (!s) return fail(DD_ERR_BAD_ARG, "null argument");
    if (nsamp_out < 0) return fail(DD_ERR_BAD_ARG, "nsamp_out must be >= 0");
    if (s->ndm == 0 || nsamp_out == 0) return DD_OK;
    if (!X || !D) return fail(DD_ERR_BAD_ARG, "X or D is null");
    if (in_stride < nsamp_out + s->ms1 + s->ms2)
        return fail(DD_ERR_BAD_ARG, "in_stride is shorter than nsamp_out + dd_subband_max_shift");
    if (out_stride < nsamp_out) return fail(DD_ERR_BAD_ARG, "out_stride is shorter than nsamp_out");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // intermediate S [subband][nominal DM][n1]: the reduced filterbanks of step 2, rows 16-byte aligned
    const int64_t n1 = nsamp_out + s->ms2, pitch = (n1 + 63) / 64 * 64;
    float* S = nullptr;
    int rc = workspace_alloc((void**)&S, (size_t)s->nsb * s->nnom * pitch * sizeof(float), cuda_stream);
    if (rc != DD_OK) return rc;
    constexpr int K = dd_subband::kStreams;
    // fork: the internal streams wait for everything queued on the caller's stream so far
    auto fork = [&]() {
        cudaError_t e = cudaEventRecord(s->fork, st);
        for (int i = 0; i < K && e == cudaSuccess; ++i) e = cudaStreamWaitEvent(s->aux[i], s->fork, 0);
        return e;
    };
    // join: the caller's stream waits for the internal streams
    auto join = [&]() {
        cudaError_t e = cudaSuccess;
        for (int i = 0; i < K && e == cudaSuccess; ++i) {
            e = cudaEventRecord(s->join[i], s->aux[i]);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(st, s->join[i], 0);
        }
        return e;
    };
    cudaError_t ce = fork();
    for (int b = 0; b < s->nsb && rc == DD_OK && ce == cudaSuccess; ++b)
        rc = dd_execute(s->sub[b], X + (int64_t)b * s->ncs * in_stride, in_stride, 0, S + (int64_t)b * s->nnom * pitch,
                        pitch, 0, n1, 1, s->aux[b % K]);
    if (ce == cudaSuccess) ce = join();                   // (also after a failed launch: nothing is left running on S)
    if (ce == cudaSuccess && rc == DD_OK) ce = fork();
    for (int g = 0; g < s->nnom && rc == DD_OK && ce == cudaSuccess; ++g)
        rc = dd_execute(s->grp[g], S + (int64_t)g * pitch, (int64_t)s->nnom * pitch, 0,
                        D + (int64_t)g * s->nds * out_stride, out_stride, 0, nsamp_out, 1, s->aux[g % K]);
    if (ce == cudaSuccess) ce = join();
    cudaFreeAsync(S, st);
    if (ce != cudaSuccess) return fail(DD_ERR_CUDA, std::string("subband dedispersion: ") + cudaGetErrorString(ce));
    return rc;
}

}  // extern "C"
