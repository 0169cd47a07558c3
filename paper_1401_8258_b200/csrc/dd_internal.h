// Internal declarations shared by the library's translation units (NOT part of the C ABI and
// not shared with oracle/).
#pragma once

#include <cstdint>
#include <string>
#include <vector>

#include "../../include/dedisp_b200.h"

namespace dd {

// ---- error plumbing ---------------------------------------------------------------------
void set_error(const std::string& msg);
int fail(int code, const std::string& msg);

// stream-ordered workspace from the library's own pool (api.cu); free with cudaFreeAsync
int workspace_alloc(void** out, size_t bytes, void* stream);

// Raises cudaFuncAttributeMaxDynamicSharedMemorySize of kernel `func` on the current device to at
// least `bytes` (never lowers it: the attribute belongs to the function, not to a plan, so plans
// with different needs must not undo each other).  Call before every launch; cached per device.
int ensure_dyn_smem(const void* func, size_t bytes);

// ---- host delay table (plan.cpp; eq 2.2/2.3) ------------------------------
struct HostTable {
    int nchans = 0;
    int ndm = 0;
    std::vector<int32_t> order;     // order[r] = caller index of the r-th smallest DM (stable)
    std::vector<int32_t> shift;     // [ndm][nchans] in SORTED DM order (monotone in r and in c)
    int64_t maxshift = 0;
};

// Validates the arguments (DD_ERR_BAD_ARG on failure) and fills the table.
int build_host_table(int nchans, double fch1, double foff, double tsamp, const double* dm_list,
                     int ndm, HostTable* out);
// Validation + maxshift only (no table storage).
int64_t host_max_shift(int nchans, double fch1, double foff, double tsamp, const double* dm_list,
                       int ndm);

// Largest s(d_last,c) - s(d_first,c) over all tiles of `kb` consecutive sorted DMs.
int64_t max_tile_spread(const HostTable& t, int kb);

// ---- kernel launchers -----------------------------------------------------------------------
struct ExecArgs {
    const void* X;
    void* D;
    int64_t in_stride, in_beam_stride, out_stride, out_beam_stride;
    int64_t nsamp_out;
    int nbeams;
    int nchans, ndm;
    const int32_t* d_shift;         // device [ndm][nchans], sorted DM order
    const int32_t* d_order;         // device [ndm], sorted row -> caller row
    void* stream;
};

// generic channel-vector kernel; kb in {16,8,4,2,1}; max_spread = largest tile spread (samples)
int launch_generic(int dtype, int kb, int max_spread, const ExecArgs& a);
// one thread per output element (direct.cu): tiny plans, nchans * ndm <= kDirectMaxCells
constexpr int64_t kDirectMaxCells = 4096;
bool direct_args_ok(const ExecArgs& a);
int launch_direct(int dtype, const ExecArgs& a);

}  // namespace dd

struct dd_plan;
struct dd_host_ws;
struct dd_ps_plan;
struct dd_psu8_plan;

namespace dd {
// uint8 front end (front_u8.cu): the four byte-shifted copies ps_u8.cu stages from
int make_shift_copies_u8(const dd_plan* p, const ExecArgs& a, uint8_t** W_out, int64_t* wcopy_out,
                         int64_t* wpitch_out);
// float32 kernel with shared partial sums (ps_f32.cu)
int build_ps_plan(dd_plan* p);
void destroy_ps_plan(dd_plan* p);
bool ps_plan_usable(const dd_plan* p);
bool ps_args_ok(const dd_plan* p, const ExecArgs& a);
int ps_launches(const dd_plan* p, const ExecArgs& a);
int launch_ps(const dd_plan* p, const ExecArgs& a);
std::string ps_describe(const dd_plan* p);
// uint8 kernel with shared partial sums (ps_u8.cu)
int build_psu8_plan(dd_plan* p);
void destroy_psu8_plan(dd_plan* p);
bool psu8_plan_usable(const dd_plan* p);
bool psu8_args_ok(const dd_plan* p, const ExecArgs& a);
int launch_psu8(const dd_plan* p, const ExecArgs& a);
std::string psu8_describe(const dd_plan* p);
// post-processing (post.cu)
int postprocess(int dtype, const void* D, int64_t stride, int64_t beam_stride, int ndm, int64_t nsamp, int nbeams,
                const dd_post_params* prm, float* Z, int64_t z_stride, int64_t z_beam_stride, double* stats,
                dd_candidate* cand, int64_t capacity, unsigned long long* count, void* cuda_stream);
int post_launches(const dd_post_params* prm, bool want_series);
int postprocess_static(int dtype, const void* D, int64_t stride, int64_t beam_stride, int ndm, int64_t nsamp,
                       int nbeams, const dd_post_params* prm, float* Z, int64_t z_stride, int64_t z_beam_stride,
                       dd_candidate* cand, int64_t capacity, unsigned long long* count, void* cuda_stream);
// coherent beamformer (beamform.cu)
int beamform_power_u4(const uint8_t* V, int nants, int nchans, int64_t nsamp, const float* W, int nbeams, float* P,
                      int64_t out_stride, int64_t out_beam_stride, void* cuda_stream);
// the same on the tcgen05 tensor cores (beamform_tc.cu): shapes it takes, and the launch
bool beamform_tc_ok(int nants, int nbeams);
int beamform_tc_launch(const uint8_t* V, int nants, int nchans, int64_t nsamp, const float* W, int nbeams, float* P,
                       int64_t out_stride, int64_t out_beam_stride, void* cuda_stream);
// RFI mitigation (rfi.cu)
int rfi_mitigate(float* X, int nchans, int64_t nsamp, int64_t stride, int64_t beam_stride, int nbeams,
                 const dd_rfi_params* prm, double* bandpass, double* fit, double* stats, uint8_t* chan_flags,
                 uint8_t* spec_flags, void* cuda_stream);
}  // namespace dd

struct dd_plan {
    int dtype = DD_F32;
    int nchans = 0, ndm = 0;
    double fch1 = 0, foff = 0, tsamp = 0;
    dd::HostTable host;
    int device = -1;
    int32_t* d_shift = nullptr;
    int32_t* d_order = nullptr;
    int kernel_pref = DD_KERNEL_AUTO;
    bool tiny = false;                  // nchans * ndm <= kDirectMaxCells: AUTO takes the direct kernel
    int generic_kb = 1;
    int generic_spread = 0;
    dd_ps_plan* ps = nullptr;           // null: the float32 partial-sum kernel does not take this plan
    dd_psu8_plan* psu8 = nullptr;       // null: the uint8 partial-sum kernel does not take this plan
    std::string ps_why;                 // why the partial-sum kernel does not take this plan (dd_plan_describe)
    dd_host_ws* host_ws = nullptr;      // device buffers / streams cached by dd_execute_host
};
