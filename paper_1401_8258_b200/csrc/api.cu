// C-ABI entry points (include/dedisp_b200.h): argument checking, plan / stream objects, kernel
// selection.  No arithmetic of the method lives here except through plan.cpp (the delay table)
// and the kernels.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>
#include <mutex>
#include <new>

#include "dd_internal.h"
#include "ps_host.h"

namespace dd {

static thread_local std::string g_last_error;

void set_error(const std::string& msg) { g_last_error = msg; }
int fail(int code, const std::string& msg)
{
    g_last_error = msg;
    return code;
}

static int cuda_fail(const char* what, cudaError_t e)
{
    return fail(DD_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define DD_CUDA(call)                                           \
    do {                                                        \
        cudaError_t e__ = (call);                               \
        if (e__ != cudaSuccess) return cuda_fail(#call, e__);   \
    } while (0)

// The library is sm_100a only: refuse anything else loudly (no CPU fallback, north_star).
static int require_sm100(int* device_out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(DD_ERR_UNSUPPORTED, std::string("no usable CUDA device: ") + cudaGetErrorString(e));
    }
    int major = 0;
    e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return cuda_fail("cudaDeviceGetAttribute", e);
    if (major != 10)
        return fail(DD_ERR_UNSUPPORTED, "device is not sm_100 (B200); this library has no other path");
    if (device_out) *device_out = dev;
    return DD_OK;
}

static size_t elem_size(int dtype) { return dtype == DD_F32 ? 4 : 1; }

// Per-call workspaces (byte-shifted copies, re-pitched input) come from a stream-ordered pool of the
// library's own that keeps its memory between calls (release threshold = max): the default pool
// would return the memory at the next synchronisation and the following call would pay for a
// fresh physical allocation.
static cudaMemPool_t pools[64] = {};
static std::mutex pools_mutex;

int workspace_alloc(void** out, size_t bytes, void* stream)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lock(pools_mutex);
    if (e == cudaSuccess && dev >= 0 && dev < 64 && !pools[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        e = cudaMemPoolCreate(&pool, &props);
        if (e == cudaSuccess) {
            uint64_t keep = UINT64_MAX;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
            pools[dev] = pool;
        }
    }
    if (e == cudaSuccess && dev >= 0 && dev < 64 && pools[dev])
        e = cudaMallocFromPoolAsync(out, bytes, pools[dev], (cudaStream_t)stream);
    else if (e == cudaSuccess)
        e = cudaMallocAsync(out, bytes, (cudaStream_t)stream);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(DD_ERR_NOMEM, std::string("workspace allocation: ") + cudaGetErrorString(e));
    }
    return DD_OK;
}

int ensure_dyn_smem(const void* func, size_t bytes)
{
    struct Key { const void* f; int dev; size_t have; };
    static std::vector<Key> cache;
    static std::mutex m;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail("cudaGetDevice", e);
    std::lock_guard<std::mutex> lock(m);
    Key* k = nullptr;
    for (Key& c : cache)
        if (c.f == func && c.dev == dev) k = &c;
    if (k && k->have >= bytes) return DD_OK;
    e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return cuda_fail("cudaFuncSetAttribute(MaxDynamicSharedMemorySize)", e);
    }
    if (k) k->have = bytes;
    else cache.push_back({func, dev, bytes});
    return DD_OK;
}

}  // namespace dd

using namespace dd;

// host-call workspace cached in the plan (see dd_execute_host)
struct dd_host_ws {
    void* dX = nullptr;
    void* dD = nullptr;
    size_t x_bytes = 0, d_bytes = 0;
    cudaStream_t s_in = nullptr, s_run = nullptr, s_out = nullptr;
    std::vector<cudaEvent_t> ev_in, ev_run;
};

struct dd_stream {
    const dd_plan* plan = nullptr;
    int64_t max_chunk = 0;
    int nbeams = 1;
    int64_t cap = 0;        // row length of the work buffers (elements), multiple of 64
    int64_t have = 0;       // samples currently held per channel (the carry)
    int64_t total_in = 0, total_out = 0;
    void* buf[2] = {nullptr, nullptr};
    int cur = 0;
};

extern "C" {

const char* dd_strerror(int code)
{
    switch (code) {
        case DD_OK: return "ok";
        case DD_ERR_BAD_ARG: return "bad argument";
        case DD_ERR_UNSUPPORTED: return "unsupported (needs an sm_100 / B200 device)";
        case DD_ERR_NOMEM: return "out of memory";
        case DD_ERR_CUDA: return "CUDA runtime error";
        case DD_ERR_STATE: return "invalid state";
    }
    return "unknown error";
}

const char* dd_last_error(void) { return g_last_error.c_str(); }
const char* dd_version(void) { return "dedisp_b200 0.1 (sm_100a)"; }

int64_t dd_max_shift(int nchans, double fch1, double foff, double tsamp, const double* dm_list, int ndm)
{
    return host_max_shift(nchans, fch1, foff, tsamp, dm_list, ndm);
}

int dd_shift_table(int nchans, double fch1, double foff, double tsamp, const double* dm_list, int ndm,
                   int32_t* host_out)
{
    if (ndm > 0 && !host_out) return fail(DD_ERR_BAD_ARG, "host_out is null");
    HostTable t;
    int rc = build_host_table(nchans, fch1, foff, tsamp, dm_list, ndm, &t);
    if (rc != DD_OK) return rc;
    for (int r = 0; r < ndm; ++r)
        std::memcpy(host_out + (size_t)t.order[r] * nchans, &t.shift[(size_t)r * nchans],
                    (size_t)nchans * sizeof(int32_t));
    return DD_OK;
}

// ------------------------------------------------------------------------------ plan

int dd_plan_create(dd_plan** out, int dtype, int nchans, double fch1, double foff, double tsamp,
                   const double* dm_list, int ndm)
{
    if (!out) return fail(DD_ERR_BAD_ARG, "out is null");
    *out = nullptr;
    if (dtype != DD_F32 && dtype != DD_U8) return fail(DD_ERR_BAD_ARG, "dtype must be DD_F32 or DD_U8");
    dd_plan* p = new (std::nothrow) dd_plan;
    if (!p) return fail(DD_ERR_NOMEM, "plan allocation failed");
    p->dtype = dtype;
    p->nchans = nchans;
    p->ndm = ndm;
    p->fch1 = fch1;
    p->foff = foff;
    p->tsamp = tsamp;
    int rc = build_host_table(nchans, fch1, foff, tsamp, dm_list, ndm, &p->host);
    if (rc != DD_OK) {
        delete p;
        return rc;
    }
    rc = require_sm100(&p->device);
    if (rc != DD_OK) {
        delete p;
        return rc;
    }
    p->tiny = (int64_t)nchans * ndm <= kDirectMaxCells;
    // generic kernel tiling: the most trials per block whose channel vector still fits
    p->generic_kb = 1;
    p->generic_spread = 0;
    const int cands[] = {16, 8, 4, 2};
    for (int kb : cands) {
        int64_t sp = max_tile_spread(p->host, kb);
        if (sp <= 512) {
            p->generic_kb = kb;
            p->generic_spread = (int)sp;
            break;
        }
    }
    if (ndm > 0) {
        cudaError_t e = cudaMalloc(&p->d_shift, p->host.shift.size() * sizeof(int32_t));
        if (e == cudaSuccess) e = cudaMalloc(&p->d_order, (size_t)ndm * sizeof(int32_t));
        if (e != cudaSuccess) {
            dd_plan_destroy(p);
            cudaGetLastError();
            return fail(DD_ERR_NOMEM, std::string("device table allocation: ") + cudaGetErrorString(e));
        }
        e = cudaMemcpy(p->d_shift, p->host.shift.data(), p->host.shift.size() * sizeof(int32_t),
                       cudaMemcpyHostToDevice);
        if (e == cudaSuccess)
            e = cudaMemcpy(p->d_order, p->host.order.data(), (size_t)ndm * sizeof(int32_t),
                           cudaMemcpyHostToDevice);
        if (e != cudaSuccess) {
            dd_plan_destroy(p);
            return cuda_fail("table upload", e);
        }
    }
    rc = build_ps_plan(p);
    if (rc == DD_OK) rc = build_psu8_plan(p);
    if (rc != DD_OK) {
        dd_plan_destroy(p);
        return rc;
    }
    *out = p;
    return DD_OK;
}

void dd_plan_destroy(dd_plan* p)
{
    if (!p) return;
    if (p->host_ws) {
        dd_host_ws* w = p->host_ws;
        if (w->dX) cudaFree(w->dX);
        if (w->dD) cudaFree(w->dD);
        for (auto e : w->ev_in) cudaEventDestroy(e);
        for (auto e : w->ev_run) cudaEventDestroy(e);
        if (w->s_in) cudaStreamDestroy(w->s_in);
        if (w->s_run) cudaStreamDestroy(w->s_run);
        if (w->s_out) cudaStreamDestroy(w->s_out);
        delete w;
    }
    destroy_ps_plan(p);
    destroy_psu8_plan(p);
    if (p->d_shift) cudaFree(p->d_shift);
    if (p->d_order) cudaFree(p->d_order);
    delete p;
}

int64_t dd_plan_max_shift(const dd_plan* p)
{
    if (!p) return fail(DD_ERR_BAD_ARG, "plan is null");
    return p->host.maxshift;
}
int dd_plan_ndm(const dd_plan* p) { return p ? p->ndm : fail(DD_ERR_BAD_ARG, "plan is null"); }
int dd_plan_nchans(const dd_plan* p) { return p ? p->nchans : fail(DD_ERR_BAD_ARG, "plan is null"); }

int dd_plan_shift_table(const dd_plan* p, int32_t* host_out)
{
    if (!p || !host_out) return fail(DD_ERR_BAD_ARG, "null argument");
    for (int r = 0; r < p->ndm; ++r)
        std::memcpy(host_out + (size_t)p->host.order[r] * p->nchans,
                    &p->host.shift[(size_t)r * p->nchans], (size_t)p->nchans * sizeof(int32_t));
    return DD_OK;
}

int dd_plan_set_kernel(dd_plan* p, int kernel)
{
    if (!p) return fail(DD_ERR_BAD_ARG, "plan is null");
    if (kernel != DD_KERNEL_AUTO && kernel != DD_KERNEL_GENERIC && kernel != DD_KERNEL_PS &&
        kernel != DD_KERNEL_DIRECT)
        return fail(DD_ERR_BAD_ARG, "unknown kernel id");
    if (kernel == DD_KERNEL_PS && !ps_plan_usable(p) && !psu8_plan_usable(p))
        return fail(DD_ERR_UNSUPPORTED, "the partial-sum kernel does not take this plan (dtype or per-trial delay steps)");
    p->kernel_pref = kernel;
    return DD_OK;
}

// The plan's tables, descriptors and workspaces live on the device it was created on.
static int check_device(const dd_plan* p)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail("cudaGetDevice", e);
    if (dev != p->device)
        return fail(DD_ERR_STATE, "the current CUDA device (" + std::to_string(dev) + ") is not the plan's device (" +
                                      std::to_string(p->device) + ")");
    return DD_OK;
}

static void fill_args(const dd_plan* p, ExecArgs* a, const void* X, int64_t in_stride, int64_t in_beam_stride,
                      void* D, int64_t out_stride, int64_t out_beam_stride, int64_t nsamp_out, int nbeams,
                      void* cuda_stream)
{
    a->X = X;
    a->D = D;
    a->in_stride = in_stride;
    a->in_beam_stride = nbeams > 1 ? in_beam_stride : 0;
    a->out_stride = out_stride;
    a->out_beam_stride = nbeams > 1 ? out_beam_stride : 0;
    a->nsamp_out = nsamp_out;
    a->nbeams = nbeams;
    a->nchans = p->nchans;
    a->ndm = p->ndm;
    a->d_shift = p->d_shift;
    a->d_order = p->d_order;
    a->stream = cuda_stream;
}

static int kernel_for(const dd_plan* p, const ExecArgs& a)
{
    if (p->kernel_pref == DD_KERNEL_GENERIC) return DD_KERNEL_GENERIC;
    if (p->kernel_pref == DD_KERNEL_DIRECT) return direct_args_ok(a) ? DD_KERNEL_DIRECT : DD_KERNEL_GENERIC;
    // tiny plans: decided from the plan alone, so every call of the plan adds in the same order
    if (p->kernel_pref == DD_KERNEL_AUTO && p->tiny && direct_args_ok(a)) return DD_KERNEL_DIRECT;
    if (psu8_plan_usable(p) && psu8_args_ok(p, a)) return DD_KERNEL_PS;
    if (ps_plan_usable(p) && ps_args_ok(p, a)) return DD_KERNEL_PS;
    return DD_KERNEL_GENERIC;
}

int dd_plan_kernel_for(const dd_plan* p, const void* X, int64_t in_stride, int64_t in_beam_stride,
                       const void* D, int64_t out_stride, int64_t out_beam_stride, int64_t nsamp_out,
                       int nbeams)
{
    if (!p) return fail(DD_ERR_BAD_ARG, "plan is null");
    if (nbeams < 1 || nsamp_out < 0) return fail(DD_ERR_BAD_ARG, "bad nbeams / nsamp_out");
    ExecArgs a;
    fill_args(p, &a, X, in_stride, in_beam_stride, const_cast<void*>(D), out_stride, out_beam_stride,
              nsamp_out, nbeams, nullptr);
    return kernel_for(p, a);
}

int dd_plan_launches_for(const dd_plan* p, const void* X, int64_t in_stride, int64_t in_beam_stride,
                         const void* D, int64_t out_stride, int64_t out_beam_stride, int64_t nsamp_out,
                         int nbeams)
{
    if (!p) return fail(DD_ERR_BAD_ARG, "plan is null");
    if (nbeams < 1 || nsamp_out < 0) return fail(DD_ERR_BAD_ARG, "bad nbeams / nsamp_out");
    if (p->ndm == 0 || nsamp_out == 0) return 0;
    ExecArgs a;
    fill_args(p, &a, X, in_stride, in_beam_stride, const_cast<void*>(D), out_stride, out_beam_stride,
              nsamp_out, nbeams, nullptr);
    if (kernel_for(p, a) != DD_KERNEL_PS) return 1;       // generic kernel: one launch
    // uint8: byte-shift front end + dedispersion kernel; float32: one launch when the input is staged
    // straight from the caller's buffer, two when it has to be re-pitched first
    return p->dtype == DD_U8 ? 2 : ps_launches(p, a);
}

int dd_execute(const dd_plan* p, const void* X, int64_t in_stride, int64_t in_beam_stride, void* D,
               int64_t out_stride, int64_t out_beam_stride, int64_t nsamp_out, int nbeams,
               void* cuda_stream)
{
    if (!p) return fail(DD_ERR_BAD_ARG, "plan is null");
    if (nsamp_out < 0) return fail(DD_ERR_BAD_ARG, "nsamp_out must be >= 0");
    if (nbeams < 1) return fail(DD_ERR_BAD_ARG, "nbeams must be >= 1");
    if (p->ndm == 0 || nsamp_out == 0) return DD_OK;
    if (!X || !D) return fail(DD_ERR_BAD_ARG, "X or D is null");
    if (in_stride < nsamp_out + p->host.maxshift)
        return fail(DD_ERR_BAD_ARG, "in_stride is shorter than nsamp_out + maxshift");
    if (out_stride < nsamp_out) return fail(DD_ERR_BAD_ARG, "out_stride is shorter than nsamp_out");
    {
        int rc = check_device(p);
        if (rc != DD_OK) return rc;
    }
    if (nbeams > 1 && (in_beam_stride <= 0 || out_beam_stride <= 0))
        return fail(DD_ERR_BAD_ARG, "beam strides must be positive when nbeams > 1");
    if (p->dtype == DD_F32 && (((uintptr_t)X | (uintptr_t)D) & 3))
        return fail(DD_ERR_BAD_ARG, "float32 buffers must be 4-byte aligned");
    if (p->dtype == DD_U8 && ((uintptr_t)D & 3))
        return fail(DD_ERR_BAD_ARG, "int32 output must be 4-byte aligned");

    ExecArgs a;
    fill_args(p, &a, X, in_stride, in_beam_stride, D, out_stride, out_beam_stride, nsamp_out, nbeams,
              cuda_stream);
    const int k = kernel_for(p, a);
    if (p->kernel_pref == DD_KERNEL_PS && k != DD_KERNEL_PS)
        return fail(DD_ERR_UNSUPPORTED, "partial-sum kernel forced but the grid does not fit");
    if (p->kernel_pref == DD_KERNEL_DIRECT && k != DD_KERNEL_DIRECT)
        return fail(DD_ERR_UNSUPPORTED, "direct kernel forced but the grid does not fit");
    if (k == DD_KERNEL_DIRECT) return launch_direct(p->dtype, a);
    if (k == DD_KERNEL_PS) return p->dtype == DD_U8 ? launch_psu8(p, a) : launch_ps(p, a);
    return launch_generic(p->dtype, p->generic_kb, p->generic_spread, a);
}

int dd_release_workspaces(void)
{
    std::lock_guard<std::mutex> lock(pools_mutex);
    for (int d = 0; d < 64; ++d)
        if (pools[d]) {
            cudaError_t e = cudaMemPoolTrimTo(pools[d], 0);
            if (e != cudaSuccess) return cuda_fail("cudaMemPoolTrimTo", e);
        }
    return DD_OK;
}

int dd_plan_describe(const dd_plan* p, char* buf, int buflen)
{
    if (!p || !buf || buflen < 1) return fail(DD_ERR_BAD_ARG, "null argument");
    std::string t = std::string(p->dtype == DD_U8 ? "uint8->int32" : "float32") + ", " + std::to_string(p->nchans) +
                    " channels x " + std::to_string(p->ndm) + " trials, maxshift " +
                    std::to_string(p->host.maxshift) + ", device " + std::to_string(p->device) + "; ";
    if (p->ndm == 0) t += "empty plan (nothing to launch)";
    else if (p->tiny && p->kernel_pref == DD_KERNEL_AUTO)
        t += "direct kernel dd_direct_kernel (tiny plan: nchans * ndm <= " + std::to_string(kDirectMaxCells) +
             ", one thread per output sample)";
    else if (p->dtype == DD_U8) t += psu8_plan_usable(p) ? psu8_describe(p) : "partial-sum kernel unavailable: " + p->ps_why;
    else t += ps_plan_usable(p) ? ps_describe(p) : "partial-sum kernel unavailable: " + p->ps_why;
    if (p->ndm > 0) t += "; generic kernel: " + std::to_string(p->generic_kb) + " trials per block";
    if (p->kernel_pref != DD_KERNEL_AUTO)
        t += std::string("; forced: ") + (p->kernel_pref == DD_KERNEL_PS ? "ps" : p->kernel_pref == DD_KERNEL_DIRECT ? "direct" : "generic");
    const int n = (int)std::min<size_t>(t.size(), (size_t)buflen - 1);
    std::memcpy(buf, t.data(), (size_t)n);
    buf[n] = 0;
    return (int)t.size();
}

// ------------------------------------------------------------------------------ one-shot

static int one_shot(int dtype, const void* X, int nchans, int64_t nsamp, double fch1, double foff,
                    double tsamp, const double* dm_list, int ndm, void* D)
{
    if (nsamp < 0) return fail(DD_ERR_BAD_ARG, "nsamp must be >= 0");
    dd_plan* p = nullptr;
    int rc = dd_plan_create(&p, dtype, nchans, fch1, foff, tsamp, dm_list, ndm);
    if (rc != DD_OK) return rc;
    rc = dd_execute(p, X, nsamp + p->host.maxshift, 0, D, nsamp, 0, nsamp, 1, nullptr);
    if (rc == DD_OK) {
        cudaError_t e = cudaStreamSynchronize(nullptr);
        if (e != cudaSuccess) rc = cuda_fail("cudaStreamSynchronize", e);
    }
    dd_plan_destroy(p);
    return rc;
}

int dd_dedisperse_f32(const float* X, int nchans, int64_t nsamp, double fch1, double foff, double tsamp,
                      const double* dm_list, int ndm, float* D)
{
    return one_shot(DD_F32, X, nchans, nsamp, fch1, foff, tsamp, dm_list, ndm, D);
}

int dd_dedisperse_u8_i32(const uint8_t* X, int nchans, int64_t nsamp, double fch1, double foff,
                         double tsamp, const double* dm_list, int ndm, int32_t* D)
{
    return one_shot(DD_U8, X, nchans, nsamp, fch1, foff, tsamp, dm_list, ndm, D);
}

// ------------------------------------------------------------------------------ host buffers

static int64_t round_up(int64_t v, int64_t m) { return (v + m - 1) / m * m; }

// Upload X in time slices, dedisperse every slice into the plan's cached device buffer and, when D is not
// null, download the slices; the three overlap on internal streams.  With D == null the result stays on the
// device (dd_search_host post-processes it there): *dD_out, *dstride_out, *dbeam_out describe it, and the
// caller continues on w->s_run.  All streams are drained before returning when D != null or on failure.
static int host_pipeline(dd_plan* p, const void* X, int64_t in_stride, int64_t in_beam_stride, void* D,
                         int64_t out_stride, int64_t out_beam_stride, int64_t nsamp_out, int nbeams,
                         void** dD_out, int64_t* dstride_out_p, int64_t* dbeam_out_p)
{
    if (!p) return fail(DD_ERR_BAD_ARG, "plan is null");
    if (nsamp_out < 0) return fail(DD_ERR_BAD_ARG, "nsamp_out must be >= 0");
    if (nbeams < 1) return fail(DD_ERR_BAD_ARG, "nbeams must be >= 1");
    if (p->ndm == 0 || nsamp_out == 0) return DD_OK;
    if (!X) return fail(DD_ERR_BAD_ARG, "X is null");
    const int64_t ms = p->host.maxshift;
    if (in_stride < nsamp_out + ms) return fail(DD_ERR_BAD_ARG, "in_stride is shorter than nsamp_out + maxshift");
    if (D && out_stride < nsamp_out) return fail(DD_ERR_BAD_ARG, "out_stride is shorter than nsamp_out");
    if (nbeams > 1 && (in_beam_stride < (int64_t)p->nchans * in_stride ||
                       (D && out_beam_stride < (int64_t)p->ndm * out_stride)))
        return fail(DD_ERR_BAD_ARG, "beam strides are shorter than a beam");
    {
        int rc = check_device(p);
        if (rc != DD_OK) return rc;
    }
    const size_t es = elem_size(p->dtype);
    const int64_t dstride_in = round_up(nsamp_out + ms, 64);
    const int64_t dstride_out = round_up(nsamp_out, 64);
    const int64_t dbeam_in = (int64_t)p->nchans * dstride_in, dbeam_out = (int64_t)p->ndm * dstride_out;
    const size_t xb = (size_t)nbeams * dbeam_in * es;
    const size_t db = (size_t)nbeams * dbeam_out * 4;

    if (!p->host_ws) {
        p->host_ws = new (std::nothrow) dd_host_ws;
        if (!p->host_ws) return fail(DD_ERR_NOMEM, "workspace allocation failed");
        dd_host_ws* w = p->host_ws;
        DD_CUDA(cudaStreamCreateWithFlags(&w->s_in, cudaStreamNonBlocking));
        DD_CUDA(cudaStreamCreateWithFlags(&w->s_run, cudaStreamNonBlocking));
        DD_CUDA(cudaStreamCreateWithFlags(&w->s_out, cudaStreamNonBlocking));
    }
    dd_host_ws* w = p->host_ws;
    if (w->x_bytes < xb) {
        if (w->dX) cudaFree(w->dX);
        w->dX = nullptr;
        w->x_bytes = 0;
        cudaError_t e = cudaMalloc(&w->dX, xb);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return fail(DD_ERR_NOMEM, std::string("device X buffer: ") + cudaGetErrorString(e));
        }
        w->x_bytes = xb;
    }
    if (w->d_bytes < db) {
        if (w->dD) cudaFree(w->dD);
        w->dD = nullptr;
        w->d_bytes = 0;
        cudaError_t e = cudaMalloc(&w->dD, db);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return fail(DD_ERR_NOMEM, std::string("device D buffer: ") + cudaGetErrorString(e));
        }
        w->d_bytes = db;
    }

    // time slices: copy-in of slice k+1 and copy-out of slice k-1 overlap the kernel of slice k; what does not
    // overlap is the upload of the first slice (plus maxshift columns) and the download of the last one, so the
    // float32 path takes 16 slices (config 3: 194.9 -> 185 ms); the uint8 path stays at 8 because its front end
    // re-forms the byte-shifted copies of the maxshift overlap for every slice
    const int target = p->dtype == DD_F32 ? 16 : 8;
    int64_t slice = round_up(std::max<int64_t>((nsamp_out + target - 1) / target, 8192), 1024);
    const int nslices = (int)((nsamp_out + slice - 1) / slice);
    while ((int)w->ev_in.size() < nslices) {
        cudaEvent_t a, b;
        DD_CUDA(cudaEventCreateWithFlags(&a, cudaEventDisableTiming));
        DD_CUDA(cudaEventCreateWithFlags(&b, cudaEventDisableTiming));
        w->ev_in.push_back(a);
        w->ev_run.push_back(b);
    }
    // After the first enqueue no path may return before the three streams have drained: the async
    // copies reference the caller's X and D.
    int rc = DD_OK;
    auto cuda_ok = [&](cudaError_t e, const char* what) {
        if (e != cudaSuccess && rc == DD_OK) rc = cuda_fail(what, e);
        return e == cudaSuccess;
    };
    int64_t in_done = 0;   // input columns already uploaded
    for (int k = 0; k < nslices && rc == DD_OK; ++k) {
        const int64_t ta = (int64_t)k * slice, tb = std::min(nsamp_out, ta + slice);
        const int64_t in_end = tb + ms;
        if (in_end > in_done) {
            for (int b = 0; b < nbeams && rc == DD_OK; ++b)
                cuda_ok(cudaMemcpy2DAsync((char*)w->dX + ((size_t)b * dbeam_in + in_done) * es, dstride_in * es,
                                          (const char*)X + ((size_t)b * in_beam_stride + in_done) * es,
                                          in_stride * es, (size_t)(in_end - in_done) * es, p->nchans,
                                          cudaMemcpyHostToDevice, w->s_in),
                        "cudaMemcpy2DAsync(H2D)");
            in_done = in_end;
        }
        if (rc != DD_OK) break;
        if (!cuda_ok(cudaEventRecord(w->ev_in[k], w->s_in), "cudaEventRecord")) break;
        if (!cuda_ok(cudaStreamWaitEvent(w->s_run, w->ev_in[k], 0), "cudaStreamWaitEvent")) break;
        const int erc = dd_execute(p, (const char*)w->dX + ta * es, dstride_in, dbeam_in, (char*)w->dD + ta * 4,
                                   dstride_out, dbeam_out, tb - ta, nbeams, w->s_run);
        if (erc != DD_OK) {
            rc = erc;
            break;
        }
        if (!D) continue;                                   // the result stays on the device
        if (!cuda_ok(cudaEventRecord(w->ev_run[k], w->s_run), "cudaEventRecord")) break;
        if (!cuda_ok(cudaStreamWaitEvent(w->s_out, w->ev_run[k], 0), "cudaStreamWaitEvent")) break;
        for (int b = 0; b < nbeams && rc == DD_OK; ++b)
            cuda_ok(cudaMemcpy2DAsync((char*)D + ((size_t)b * out_beam_stride + ta) * 4, out_stride * 4,
                                      (const char*)w->dD + ((size_t)b * dbeam_out + ta) * 4, dstride_out * 4,
                                      (size_t)(tb - ta) * 4, p->ndm, cudaMemcpyDeviceToHost, w->s_out),
                    "cudaMemcpy2DAsync(D2H)");
    }
    if (dD_out) {
        *dD_out = w->dD;
        *dstride_out_p = dstride_out;
        *dbeam_out_p = dbeam_out;
    }
    if (D || rc != DD_OK) {
        const std::string first_error = rc != DD_OK ? g_last_error : std::string();
        cuda_ok(cudaStreamSynchronize(w->s_out), "cudaStreamSynchronize");
        cuda_ok(cudaStreamSynchronize(w->s_run), "cudaStreamSynchronize");
        cuda_ok(cudaStreamSynchronize(w->s_in), "cudaStreamSynchronize");
        if (!first_error.empty()) g_last_error = first_error;
    }
    return rc;
}

int dd_execute_host(dd_plan* p, const void* X, int64_t in_stride, int64_t in_beam_stride, void* D,
                    int64_t out_stride, int64_t out_beam_stride, int64_t nsamp_out, int nbeams)
{
    if (p && p->ndm > 0 && nsamp_out > 0 && !D) return fail(DD_ERR_BAD_ARG, "X or D is null");
    return host_pipeline(p, X, in_stride, in_beam_stride, D, out_stride, out_beam_stride, nsamp_out, nbeams,
                         nullptr, nullptr, nullptr);
}

// ------------------------------------------------------------------------------ post-processing

int dd_postprocess(int dtype, const void* D, int64_t stride, int64_t beam_stride, int ndm, int64_t nsamp,
                   int nbeams, const dd_post_params* params, float* Z, int64_t z_stride, int64_t z_beam_stride,
                   double* stats, dd_candidate* cand, int64_t capacity, unsigned long long* count,
                   void* cuda_stream)
{
    int rc = require_sm100(nullptr);
    if (rc != DD_OK) return rc;
    return postprocess(dtype, D, stride, beam_stride, ndm, nsamp, nbeams, params, Z, z_stride, z_beam_stride, stats,
                       cand, capacity, count, cuda_stream);
}

int dd_postprocess_static(int dtype, const void* D, int64_t stride, int64_t beam_stride, int ndm, int64_t nsamp,
                          int nbeams, const dd_post_params* params, float* Z, int64_t z_stride,
                          int64_t z_beam_stride, dd_candidate* cand, int64_t capacity, unsigned long long* count,
                          void* cuda_stream)
{
    int rc = require_sm100(nullptr);
    if (rc != DD_OK) return rc;
    return postprocess_static(dtype, D, stride, beam_stride, ndm, nsamp, nbeams, params, Z, z_stride, z_beam_stride,
                              cand, capacity, count, cuda_stream);
}

int dd_postprocess_launches(const dd_post_params* params, int want_series)
{
    if (!params) return fail(DD_ERR_BAD_ARG, "params is null");
    return post_launches(params, want_series != 0);
}

int dd_rfi_mitigate(float* X, int nchans, int64_t nsamp, int64_t stride, int64_t beam_stride, int nbeams,
                    const dd_rfi_params* params, double* bandpass, double* fit, double* stats, uint8_t* chan_flags,
                    uint8_t* spec_flags, void* cuda_stream)
{
    int rc = require_sm100(nullptr);
    if (rc != DD_OK) return rc;
    return rfi_mitigate(X, nchans, nsamp, stride, beam_stride, nbeams, params, bandpass, fit, stats, chan_flags,
                        spec_flags, cuda_stream);
}

int dd_beamform_power_u4(const uint8_t* V, int nants, int nchans, int64_t nsamp, const float* W, int nbeams, float* P,
                         int64_t out_stride, int64_t out_beam_stride, void* cuda_stream)
{
    int rc = require_sm100(nullptr);
    if (rc != DD_OK) return rc;
    return beamform_power_u4(V, nants, nchans, nsamp, W, nbeams, P, out_stride, out_beam_stride, cuda_stream);
}

int dd_search_host(dd_plan* p, const void* X, int64_t in_stride, int64_t in_beam_stride, int64_t nsamp_out,
                   int nbeams, const dd_post_params* params, dd_candidate* cand, int64_t capacity, int64_t* count)
{
    if (!p || !params || !count) return fail(DD_ERR_BAD_ARG, "null argument");
    *count = 0;
    if (!params->threshold_on) return fail(DD_ERR_BAD_ARG, "dd_search_host needs params->threshold_on");
    if (capacity < 0 || (capacity > 0 && !cand)) return fail(DD_ERR_BAD_ARG, "bad candidate buffer");
    if (p->ndm == 0 || nsamp_out == 0) return DD_OK;
    void* dD = nullptr;
    int64_t dstride = 0, dbeam = 0;
    int rc = host_pipeline(p, X, in_stride, in_beam_stride, nullptr, 0, 0, nsamp_out, nbeams, &dD, &dstride, &dbeam);
    if (rc != DD_OK) return rc;
    dd_host_ws* w = p->host_ws;
    // candidates and the counter: one stream-ordered workspace, [counter (16 bytes)][capacity entries]
    char* ws = nullptr;
    const size_t bytes = 16 + (size_t)capacity * sizeof(dd_candidate);
    rc = workspace_alloc((void**)&ws, bytes, w->s_run);
    if (rc == DD_OK) {
        cudaError_t e = cudaMemsetAsync(ws, 0, 16, w->s_run);
        if (e != cudaSuccess) rc = cuda_fail("cudaMemsetAsync", e);
    }
    if (rc == DD_OK)
        rc = postprocess(p->dtype, dD, dstride, dbeam, p->ndm, nsamp_out, nbeams, params, nullptr, 0, 0, nullptr,
                         (dd_candidate*)(ws + 16), capacity, (unsigned long long*)ws, w->s_run);
    unsigned long long n = 0;
    if (rc == DD_OK) {
        cudaError_t e = cudaMemcpyAsync(&n, ws, sizeof(n), cudaMemcpyDeviceToHost, w->s_run);
        if (e == cudaSuccess) e = cudaStreamSynchronize(w->s_run);
        if (e != cudaSuccess) rc = cuda_fail("candidate count download", e);
    }
    if (rc == DD_OK && n > 0 && capacity > 0) {
        const size_t k = (size_t)std::min<unsigned long long>(n, (unsigned long long)capacity);
        cudaError_t e = cudaMemcpyAsync(cand, ws + 16, k * sizeof(dd_candidate), cudaMemcpyDeviceToHost, w->s_run);
        if (e != cudaSuccess) rc = cuda_fail("candidate download", e);
    }
    if (ws) cudaFreeAsync(ws, w->s_run);
    cudaError_t e = cudaStreamSynchronize(w->s_run);
    if (e != cudaSuccess && rc == DD_OK) rc = cuda_fail("cudaStreamSynchronize", e);
    cudaStreamSynchronize(w->s_in);
    *count = (int64_t)n;
    return rc;
}

static int one_shot_host(int dtype, const void* X, int nchans, int64_t nsamp, double fch1, double foff,
                         double tsamp, const double* dm_list, int ndm, void* D)
{
    if (nsamp < 0) return fail(DD_ERR_BAD_ARG, "nsamp must be >= 0");
    dd_plan* p = nullptr;
    int rc = dd_plan_create(&p, dtype, nchans, fch1, foff, tsamp, dm_list, ndm);
    if (rc != DD_OK) return rc;
    rc = dd_execute_host(p, X, nsamp + p->host.maxshift, 0, D, nsamp, 0, nsamp, 1);
    dd_plan_destroy(p);
    return rc;
}

int dd_dedisperse_f32_host(const float* X, int nchans, int64_t nsamp, double fch1, double foff,
                           double tsamp, const double* dm_list, int ndm, float* D)
{
    return one_shot_host(DD_F32, X, nchans, nsamp, fch1, foff, tsamp, dm_list, ndm, D);
}

int dd_dedisperse_u8_i32_host(const uint8_t* X, int nchans, int64_t nsamp, double fch1, double foff,
                              double tsamp, const double* dm_list, int ndm, int32_t* D)
{
    return one_shot_host(DD_U8, X, nchans, nsamp, fch1, foff, tsamp, dm_list, ndm, D);
}

// ------------------------------------------------------------------------------ streaming

int dd_stream_create(dd_stream** out, const dd_plan* plan, int64_t max_chunk, int nbeams)
{
    if (!out) return fail(DD_ERR_BAD_ARG, "out is null");
    *out = nullptr;
    if (!plan) return fail(DD_ERR_BAD_ARG, "plan is null");
    if (max_chunk < 1) return fail(DD_ERR_BAD_ARG, "max_chunk must be >= 1");
    if (nbeams < 1) return fail(DD_ERR_BAD_ARG, "nbeams must be >= 1");
    dd_stream* s = new (std::nothrow) dd_stream;
    if (!s) return fail(DD_ERR_NOMEM, "stream allocation failed");
    s->plan = plan;
    s->max_chunk = max_chunk;
    s->nbeams = nbeams;
    s->cap = round_up(plan->host.maxshift + max_chunk, 64);
    const size_t bytes = (size_t)nbeams * plan->nchans * s->cap * elem_size(plan->dtype);
    for (int i = 0; i < 2; ++i) {
        cudaError_t e = cudaMalloc(&s->buf[i], bytes);
        if (e != cudaSuccess) {
            cudaGetLastError();
            dd_stream_destroy(s);
            return fail(DD_ERR_NOMEM, std::string("stream work buffer: ") + cudaGetErrorString(e));
        }
    }
    *out = s;
    return DD_OK;
}

int dd_stream_push(dd_stream* s, const void* X_new, int64_t in_stride, int64_t in_beam_stride,
                   int64_t n_new, void* D_out, int64_t out_stride, int64_t out_beam_stride,
                   int64_t* n_out, void* cuda_stream)
{
    if (n_out) *n_out = 0;
    if (!s || !n_out) return fail(DD_ERR_BAD_ARG, "null argument");
    if (n_new < 0) return fail(DD_ERR_BAD_ARG, "n_new must be >= 0");
    if (n_new > s->max_chunk) return fail(DD_ERR_STATE, "n_new exceeds the stream's max_chunk");
    if (n_new == 0) return DD_OK;
    if (!X_new) return fail(DD_ERR_BAD_ARG, "X_new is null");
    if (in_stride < n_new) return fail(DD_ERR_BAD_ARG, "in_stride is shorter than n_new");
    const dd_plan* p = s->plan;
    {
        int rc = check_device(p);
        if (rc != DD_OK) return rc;
    }
    const size_t es = elem_size(p->dtype);
    const int nch = p->nchans;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (s->nbeams > 1 && in_beam_stride <= 0) return fail(DD_ERR_BAD_ARG, "in_beam_stride must be positive");

    // 1. append the new samples after the carry ("the next input buffer is copied
    //    after the shifted samples")
    char* cur = (char*)s->buf[s->cur];
    const bool packed = s->nbeams == 1 || in_beam_stride == (int64_t)nch * in_stride;
    if (packed) {
        DD_CUDA(cudaMemcpy2DAsync(cur + s->have * es, s->cap * es, X_new, in_stride * es, n_new * es,
                                  (size_t)nch * s->nbeams, cudaMemcpyDeviceToDevice, st));
    } else {
        for (int b = 0; b < s->nbeams; ++b)
            DD_CUDA(cudaMemcpy2DAsync(cur + ((size_t)b * nch * s->cap + s->have) * es, s->cap * es,
                                      (const char*)X_new + (size_t)b * in_beam_stride * es,
                                      in_stride * es, n_new * es, nch, cudaMemcpyDeviceToDevice, st));
    }
    const int64_t total = s->have + n_new;
    const int64_t emit = std::max<int64_t>(0, total - p->host.maxshift);
    // 2. every output sample whose whole sweep is present
    if (emit > 0 && p->ndm > 0) {
        if (!D_out) return fail(DD_ERR_BAD_ARG, "D_out is null");
        // the work buffer holds total = emit + maxshift valid samples; its stride is cap
        int rc = dd_execute(p, cur, s->cap, (int64_t)nch * s->cap, D_out, out_stride, out_beam_stride,
                            emit, s->nbeams, cuda_stream);
        if (rc != DD_OK) return rc;
    }
    // 3. keep the last (total - emit) <= maxshift samples of every channel at the row head
    const int64_t carry = total - emit;
    if (emit > 0) {
        char* nxt = (char*)s->buf[s->cur ^ 1];
        if (carry > 0)
            DD_CUDA(cudaMemcpy2DAsync(nxt, s->cap * es, cur + emit * es, s->cap * es, carry * es,
                                      (size_t)nch * s->nbeams, cudaMemcpyDeviceToDevice, st));
        s->cur ^= 1;
    }
    s->have = carry;
    s->total_in += n_new;
    s->total_out += emit;
    *n_out = emit;
    return DD_OK;
}

int dd_stream_reset(dd_stream* s)
{
    if (!s) return fail(DD_ERR_BAD_ARG, "stream is null");
    s->have = 0;
    s->total_in = s->total_out = 0;
    return DD_OK;
}

void dd_stream_destroy(dd_stream* s)
{
    if (!s) return;
    for (int i = 0; i < 2; ++i)
        if (s->buf[i]) cudaFree(s->buf[i]);
    delete s;
}

}  // extern "C"
