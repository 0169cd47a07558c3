/* dedisp_b200.h — C ABI of the B200-native direct incoherent dedispersion library.
 *
 * What every call computes (§2.1.1 eq 2.1-2.3; constant eq 1.14,
 * PAPER.md:425; BASELINE.json north_star):
 *
 *     D[b][d][t] = sum_{c=0}^{nchans-1} X[b][c][ t + s(d,c) ]
 *     s(d,c)     = floor( 4148.808 * DM_d * (f_c^-2 - fch1^-2) / tsamp + 0.5 )   (double)
 *     f_c        = fch1 + c*foff   [MHz],   tsamp [s],   foff <= 0  (channel 0 = top of band
 *                                                                      = reference, s(d,0)=0)
 *
 * Layouts ("stored in channel order, with time changing the fastest";
 * PAPER.md:1202 the buffer holds nsamp + maxshift spectra; PAPER.md:956 the output is
 * the (DM, t) plane; PAPER.md:1131 beams are [beam][chan][time]):
 *     X : [nbeams][nchans][>= nsamp + maxshift]   time fastest, uint8 or float32
 *     D : [nbeams][ndm][nsamp]                    time fastest, int32  or float32
 * `nsamp` is always the number of OUTPUT samples per DM trial; input rows must hold
 * nsamp + maxshift samples, maxshift = max_d s(d, nchans-1) (reading R7).
 * uint8 input is accumulated in int32 and the result is exact; float32 input is
 * accumulated in float32 in a fixed channel order that depends only on the plan
 * (never on the tile position), so batch, streaming and one-shot results are bit-identical.
 *
 * Every step runs in hand-written sm_100a CUDA kernels; there is NO CPU fallback:
 * without a usable sm_100 device the compute calls return DD_ERR_UNSUPPORTED / DD_ERR_CUDA.
 *
 * Conventions
 *   - "DEVICE" pointers are CUDA device memory owned by the caller; "HOST" pointers are
 *     ordinary (pageable or pinned) host memory owned by the caller.  The library owns only
 *     what it allocates inside dd_plan / dd_stream.  X and D must not overlap.
 *   - All functions return int (0 = DD_OK, <0 = error) unless stated otherwise; they never
 *     throw, exit or print.  dd_last_error() gives a thread-local detail string.
 *   - dd_execute / dd_stream_push enqueue work on `cuda_stream` (a cudaStream_t passed as
 *     void*, NULL = legacy default stream) and return WITHOUT synchronising.  The
 *     nine-argument dd_dedisperse_* calls and the *_host calls synchronise before returning.
 *   - Errors: DD_ERR_BAD_ARG for null pointers, nchans < 1, ndm < 0, nsamp < 0, tsamp <= 0,
 *     non-finite or negative DM, fch1 <= 0 or any f_c <= 0, foff > 0 (negative shifts),
 *     a stride shorter than the row, a shift above INT32_MAX/2.  ndm == 0 or nsamp == 0 is
 *     DD_OK and writes nothing.
 */
#ifndef DEDISP_B200_H
#define DEDISP_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    DD_OK              =  0,
    DD_ERR_BAD_ARG     = -1,
    DD_ERR_UNSUPPORTED = -2,   /* no sm_100 device, or a dtype/kernel the plan does not have */
    DD_ERR_NOMEM       = -3,
    DD_ERR_CUDA        = -4,   /* a CUDA runtime call failed; see dd_last_error() */
    DD_ERR_STATE       = -5    /* stream pushed beyond its declared max_chunk; the current CUDA device is
                                  not the one the plan was created on */
};

enum { DD_F32 = 0,   /* float32 in, float32 out  */
       DD_U8  = 1 }; /* uint8   in, int32   out  */

/* kernel selection for dd_plan_set_kernel (tests and benchmarks; default DD_KERNEL_AUTO) */
enum { DD_KERNEL_AUTO    = 0,
       DD_KERNEL_GENERIC = 1,   /* shared-memory channel-vector kernel (thesis Alg. 1 modernised), any DM list */
       DD_KERNEL_DIRECT  = 3,   /* one thread per output sample, operands straight from global memory / L2;
                                   AUTO takes it for tiny plans (nchans * ndm <= 4096), which are bound by
                                   launch latency and grid size, not by any pipe (decided from the plan
                                   alone, so all calls of a plan add in the same order); on series of
                                   1e5 samples and more DD_KERNEL_PS / DD_KERNEL_GENERIC are up to 1.8x
                                   faster for such plans: choose them with dd_plan_set_kernel */
       DD_KERNEL_PS      = 2 }; /* TMA-staged kernels (float32 and uint8) with partial sums of 4-8 adjacent
                                   channels shared between the trials of a 64/128-trial tile; plans whose
                                   per-trial delay steps are too coarse for them run DD_KERNEL_GENERIC
                                   (dd_plan_describe says which and why) */

const char* dd_strerror(int code);   /* static string for an error code */
const char* dd_last_error(void);     /* thread-local detail of the last failure ("" if none) */
const char* dd_version(void);        /* static "dedisp_b200 x.y (sm_100a)" */

/* ---- the delay table (eq 2.2/2.3), host only, double precision -------- */

/* maxshift = max over d, c of s(d,c).  dm_list: HOST, ndm doubles.  <0 = error code. */
int64_t dd_max_shift(int nchans, double fch1, double foff, double tsamp,
                     const double* dm_list, int ndm);

/* The whole table, HOST int32 [ndm][nchans] in dm_list order; no GPU needed. */
int dd_shift_table(int nchans, double fch1, double foff, double tsamp,
                   const double* dm_list, int ndm, int32_t* host_out);

/* ---- one-shot calls (north_star signature): X, D are DEVICE pointers ---------------------
 * X: [nchans][nsamp + maxshift] contiguous; D: [ndm][nsamp] contiguous, rows in dm_list order.
 * Builds a plan, runs it on the legacy default stream, synchronises, destroys the plan. */
int dd_dedisperse_f32   (const float*   X, int nchans, int64_t nsamp, double fch1, double foff,
                         double tsamp, const double* dm_list, int ndm, float*   D);
int dd_dedisperse_u8_i32(const uint8_t* X, int nchans, int64_t nsamp, double fch1, double foff,
                         double tsamp, const double* dm_list, int ndm, int32_t* D);

/* Same, with HOST X and D (pageable or pinned): the library allocates device buffers, copies
 * X up, computes, copies D back, overlapping the three in time slices.  This is the
 * end-to-end call bench.py times ("e2e"). */
int dd_dedisperse_f32_host   (const float*   X, int nchans, int64_t nsamp, double fch1, double foff,
                              double tsamp, const double* dm_list, int ndm, float*   D);
int dd_dedisperse_u8_i32_host(const uint8_t* X, int nchans, int64_t nsamp, double fch1, double foff,
                              double tsamp, const double* dm_list, int ndm, int32_t* D);

/* ---- plan form: the table is built once ("computed once during thread
 * initialisation and transferred to GPU memory") and reused ------------------------------- */
typedef struct dd_plan dd_plan;

/* dm_list: HOST; any finite non-negative values in any order (duplicates allowed); output rows
 * are written in the caller's order.  Uploads the device tables on the current device. */
int     dd_plan_create(dd_plan** out, int dtype, int nchans, double fch1, double foff,
                       double tsamp, const double* dm_list, int ndm);
void    dd_plan_destroy(dd_plan* plan);
int64_t dd_plan_max_shift(const dd_plan* plan);                 /* <0 = error */
int     dd_plan_ndm(const dd_plan* plan);
int     dd_plan_nchans(const dd_plan* plan);
/* the plan's own delay table, HOST int32 [ndm][nchans] in caller DM order (tests compare it
 * with the oracle's independently built table) */
int     dd_plan_shift_table(const dd_plan* plan, int32_t* host_out);
int     dd_plan_set_kernel(dd_plan* plan, int kernel);          /* DD_KERNEL_* */
/* which kernel dd_execute would launch for these arguments: DD_KERNEL_DIRECT (tiny plans), DD_KERNEL_PS
 * (both dtypes, whenever the plan's delay steps are fine enough for shared partial sums) or
 * DD_KERNEL_GENERIC */
int     dd_plan_kernel_for(const dd_plan* plan, const void* X, int64_t in_stride,
                           int64_t in_beam_stride, const void* D, int64_t out_stride,
                           int64_t out_beam_stride, int64_t nsamp_out, int nbeams);
/* number of kernels dd_execute launches for these arguments (bench.py's gpu_launches): 1 for the generic
 * kernel and for float32 input staged straight from the caller's buffer, 2 when a front end runs first
 * (uint8 byte-shifted copies; float32 re-pitch of input that is not 16-byte aligned); 0 for empty work */
int     dd_plan_launches_for(const dd_plan* plan, const void* X, int64_t in_stride,
                             int64_t in_beam_stride, const void* D, int64_t out_stride,
                             int64_t out_beam_stride, int64_t nsamp_out, int nbeams);
/* One line of text about the plan: shape, which kernel AUTO takes and its tile shape, or why the
 * partial-sum kernel does not take the plan (then dd_execute runs the ~4x slower generic kernel).
 * Writes at most buflen-1 characters + NUL to buf (HOST); returns the untruncated length. */
int     dd_plan_describe(const dd_plan* plan, char* buf, int buflen);

/* X, D: DEVICE.  Strides are in ELEMENTS.  in_stride >= nsamp_out + maxshift is the distance
 * between channel rows, in_beam_stride between beams (ignored if nbeams == 1); same for D.
 * Reads X[b][c][0 .. nsamp_out + s(d,c)), writes D[b][d][0 .. nsamp_out).  The current CUDA
 * device must be the one the plan was created on (else DD_ERR_STATE). */
int     dd_execute(const dd_plan* plan, const void* X, int64_t in_stride, int64_t in_beam_stride,
                   void* D, int64_t out_stride, int64_t out_beam_stride,
                   int64_t nsamp_out, int nbeams, void* cuda_stream);

/* X, D: HOST (pinned memory makes the copies asynchronous), same layout and strides as dd_execute.
 * Uploads X in time slices, runs dd_execute per slice and downloads D, the three overlapped on
 * internal streams; returns after everything has landed in D (also on failure: no copy that
 * references X or D is in flight when the call returns).  Device buffers are cached in the plan
 * between calls, so one plan must not be used by two host threads at once. */
int     dd_execute_host(dd_plan* plan, const void* X, int64_t in_stride, int64_t in_beam_stride,
                        void* D, int64_t out_stride, int64_t out_beam_stride,
                        int64_t nsamp_out, int nbeams);

/* Per-call workspaces (uint8 byte-shifted copies = 4x the input, re-pitched float32 input) come from
 * a stream-ordered memory pool owned by the library that keeps its memory between calls.  This
 * returns all unused pool memory to the driver (every device). */
int     dd_release_workspaces(void);

/* ---- streaming (the last maxshift spectra are kept at the head of the buffer
 * and the next input appended; buffer sizing eq 3.3) ------------------- */
typedef struct dd_stream dd_stream;

/* The stream keeps a device work buffer of nbeams*nchans*(maxshift + max_chunk) elements
 * (double-buffered).  The plan must outlive the stream. */
int     dd_stream_create(dd_stream** out, const dd_plan* plan, int64_t max_chunk, int nbeams);
/* X_new: DEVICE [nbeams][nchans][n_new] (strides in elements), 0 <= n_new <= max_chunk.
 * Emits into D_out (DEVICE, [nbeams][ndm][>= *n_out]) every output sample whose full sweep is
 * now available: *n_out = max(0, total_in - maxshift) - total_out_so_far.  The concatenation
 * of the emitted blocks equals the one-shot result on the concatenated input, bit for bit.
 * The append, the kernels and the carry copy are ordered on `cuda_stream` only: use ONE CUDA stream
 * per dd_stream (or synchronise between pushes made on different streams), and one host thread. */
int     dd_stream_push(dd_stream* s, const void* X_new, int64_t in_stride, int64_t in_beam_stride,
                       int64_t n_new, void* D_out, int64_t out_stride, int64_t out_beam_stride,
                       int64_t* n_out, void* cuda_stream);
int     dd_stream_reset(dd_stream* s);
void    dd_stream_destroy(dd_stream* s);

/* ---- post-processing of the dedispersed series and first stage of event detection
 * (§3.5 "Signal Post-processing", §3.6 "Detection and Candidate Selection"),
 * on the device: the (DM, t) plane stays in HBM, only the candidate list goes back to the host.
 * Steps, in the paper's order; each series (one beam, one DM trial, nsamp samples) on its own:
 *   1. median filter, eq 3.4: y_m = median{x_i, |i - m| <= (w-1)/2}, w odd ("5 or 7"), window
 *      indices clamped to the ends of the series;
 *   2. detrend: subtract the least-squares line through (t, y_t), t = 0..nsamp-1;
 *   3. normalise: divide by the population standard deviation of the detrended series (a constant
 *      series gives zeros);
 *   4. threshold: samples whose value exceeds nsigma standard deviations (strictly) become
 *      (beam, dm, t, value) candidates, value in units of sigma.
 * The regression sums, the standard deviation and the threshold comparison are evaluated in double
 * precision; medians are exact selections. */
typedef struct dd_post_params {
    int   median_window;   /* 0 or 1: no median filter; else 3, 5, 7 or 9 */
    int   detrend;         /* 1: step 2 */
    int   normalise;       /* 1: step 3 (needs detrend) */
    int   threshold_on;    /* 1: step 4 (needs detrend: sigma is that of the detrended series) */
    float nsigma;          /* threshold in units of sigma */
} dd_post_params;

typedef struct dd_candidate {
    int32_t beam;          /* beam index */
    int32_t dm;            /* DM trial: row index of D (the caller's dm_list order) */
    int32_t t;             /* output sample */
    float   value;         /* detrended sample / sigma */
} dd_candidate;

/* D: DEVICE series [nbeams][ndm][nsamp] as dd_execute wrote them -- float32 for dtype DD_F32, int32 for
 * DD_U8 -- strides in elements; not modified unless Z aliases it.
 * Z: DEVICE float32 [nbeams][ndm][nsamp] (strides z_stride, z_beam_stride) receives the processed series,
 * or NULL; Z may be D itself (same strides) only when median_window <= 1.
 * stats: DEVICE double [nbeams*ndm][3] = (intercept, slope, sigma) per series, or NULL.
 * cand / capacity / count: DEVICE candidate buffer, its size in entries, and a DEVICE counter that the
 * CALLER zeroes; the counter is advanced for every detection, entries beyond capacity are dropped
 * (count > capacity tells), the order of the entries is unspecified.  Needed when threshold_on.
 * Enqueued on cuda_stream, no synchronisation.  nsamp must fit int32. */
int     dd_postprocess(int dtype, const void* D, int64_t stride, int64_t beam_stride, int ndm,
                       int64_t nsamp, int nbeams, const dd_post_params* params,
                       float* Z, int64_t z_stride, int64_t z_beam_stride, double* stats,
                       dd_candidate* cand, int64_t capacity, unsigned long long* count,
                       void* cuda_stream);
/* dd_postprocess for callers that must not allocate device memory (CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): same steps, same kernels, same results, but the per-series statistics
 * table -- the path's only scratch memory -- is a static device array inside the library instead of a
 * workspace allocation, so the call reaches no cudaMalloc / cudaMallocAsync / cudaFree.  Arguments as
 * dd_postprocess without `stats` (the caller still passes D, Z, cand, count: all DEVICE).
 * Limits: nbeams * ndm <= DD_POSTPROCESS_STATIC_MAX_SERIES, else DD_ERR_UNSUPPORTED (nothing is enqueued).
 * The array (3 doubles per series, 384 KiB) is held by every GPU that loads the library until the process
 * exits, is shared by ALL calls on that device and keeps the last call's statistics (nothing needs to
 * start at zero: each call writes every entry it reads).  Calls that overlap on the GPU (different
 * streams, no ordering between them) race on it; calls on one stream, or ordered by events, are safe. */
#define DD_POSTPROCESS_STATIC_MAX_SERIES 16384
int     dd_postprocess_static(int dtype, const void* D, int64_t stride, int64_t beam_stride, int ndm,
                              int64_t nsamp, int nbeams, const dd_post_params* params,
                              float* Z, int64_t z_stride, int64_t z_beam_stride,
                              dd_candidate* cand, int64_t capacity, unsigned long long* count,
                              void* cuda_stream);
/* number of kernels dd_postprocess launches for these parameters (bench.py's gpu_launches) */
int     dd_postprocess_launches(const dd_post_params* params, int want_series);

/* End to end with HOST buffers: uploads X (as dd_execute_host), dedisperses into a device buffer cached in
 * the plan, post-processes it there and downloads ONLY the candidates: cand (HOST, capacity entries) and
 * *count (HOST; may exceed capacity).  params->threshold_on must be 1.  Synchronous. */
int     dd_search_host(dd_plan* plan, const void* X, int64_t in_stride, int64_t in_beam_stride,
                       int64_t nsamp_out, int nbeams, const dd_post_params* params,
                       dd_candidate* cand, int64_t capacity, int64_t* count);

/* ---- RFI mitigation front end on the input buffer, before dedispersion (§3.3),
 * in place on the device.  Stages, in the paper's order, per beam:
 *   1. averaged bandpass b_c = mean_t X[c][t]; least-squares polynomial of order poly_order through
 *      (x_c, b_c), x_c the channel index mapped onto [-1, 1]; RMSE = sqrt(mean_c (b_c - B_c)^2);
 *   2. channel thresholding (eq 3.1): every channel is cut into non-overlapping windows of `window`
 *      samples (the last may be shorter); a window with |mean - B_c| > t_chan * RMSE and its two
 *      neighbours are replaced by the fitted bandpass value B_c;
 *   3. spectrum thresholding (eq 3.2): with m_t the mean over channels of spectrum t (after step 2) and
 *      mu, sigma the mean and population standard deviation of m over time, a spectrum with
 *      m_t - mu > t_spec * sigma has (m_t - mean_c B_c) subtracted from every channel;
 *   4. B_c is subtracted from every sample (the corrected spectra sit at a mean of ~0).
 * Means, fit and comparisons are evaluated in double; the output is rounded once to float32. */
typedef struct dd_rfi_params {
    int   poly_order;      /* 0..12 ("p-th order polynomial") */
    int   window;          /* W_c, samples per channel-thresholding window (thesis test: 512) */
    float t_chan;          /* channel threshold in units of the fit's RMSE (thesis test: 7) */
    float t_spec;          /* spectrum threshold in units of sigma of the spectrum means (thesis test: 5) */
} dd_rfi_params;

/* X: DEVICE float32 [nbeams][nchans][nsamp], strides in elements, modified in place.  Optional DEVICE
 * outputs (NULL to skip): bandpass and fit, double [nbeams][nchans] (b_c and B_c); stats, double
 * [nbeams][4] = (RMSE, mean_c B_c, mu, sigma); chan_flags, uint8 [nbeams][nchans][ceil(nsamp/window)]
 * (1 = window replaced); spec_flags, uint8 [nbeams][nsamp] (1 = spectrum corrected).  At most 65535
 * channel rows (nbeams * nchans) per call.  Enqueued on cuda_stream, no synchronisation. */
int     dd_rfi_mitigate(float* X, int nchans, int64_t nsamp, int64_t stride, int64_t beam_stride, int nbeams,
                        const dd_rfi_params* params, double* bandpass, double* fit, double* stats,
                        uint8_t* chan_flags, uint8_t* spec_flags, void* cuda_stream);

/* ---- approximate variants (float32), built from the exact kernels on reduced data -----------------
 * A. Time binning: trials with DM >= 2 DM_diag run on the input summed over
 *    2^k adjacent samples, k = floor(log2(DM / DM_diag)) capped at max_level, with sampling time
 *    2^k tsamp in the delay formula; DM_diag is the DM at which the delay across the LAST channel is one
 *    sample (dd_diagonal_dm), or the caller's value.  dm_list must be non-decreasing. */
double  dd_diagonal_dm(int nchans, double fch1, double foff, double tsamp);    /* host only; inf for 1 channel */
/* Y[r][i] = X[r][2i] + X[r][2i+1], i < n_in / 2; X, Y: DEVICE float32 rows, strides in elements */
int     dd_downsample2_f32(const float* X, float* Y, int64_t nrows, int64_t n_in, int64_t stride_in,
                           int64_t stride_out, void* cuda_stream);
typedef struct dd_timebin dd_timebin;
int     dd_timebin_create(dd_timebin** out, int nchans, double fch1, double foff, double tsamp,
                          const double* dm_list, int ndm, double dm_diag /* <= 0: dd_diagonal_dm */,
                          int max_level);
void    dd_timebin_destroy(dd_timebin* t);
/* number of levels; level_of_trial (HOST int32 [ndm], may be NULL) receives k per trial */
int     dd_timebin_levels(const dd_timebin* t, int32_t* level_of_trial);
/* full-rate samples every input row must hold for nsamp_out (full-rate) output samples */
int64_t dd_timebin_input_samples(const dd_timebin* t, int64_t nsamp_out);
/* X: DEVICE [nchans][n_in] (stride in_stride); D: DEVICE [ndm][out_stride]: row d receives
 * nsamp_out >> level(d) samples, sample i covering full-rate samples [2^k i, 2^k (i+1)); the rest of
 * the row is not written. */
int     dd_timebin_execute(dd_timebin* t, const float* X, int64_t in_stride, int64_t n_in, float* D,
                           int64_t out_stride, int64_t nsamp_out, void* cuda_stream);

/* B. Subband dedispersion (§2.1.3).  Step 1: every block of chans_per_subband channels is
 *    dedispersed as a filterbank of its own (reference = its first channel) at one nominal DM per block
 *    of dms_per_nominal consecutive trials (the block's middle trial).  Step 2: for every nominal DM the
 *    subband series form a filterbank of ceil(nchans / chans_per_subband) channels (fch1' = fch1,
 *    foff' = chans_per_subband * foff) that is dedispersed at each trial of the block.  dm_list must be
 *    non-decreasing.  Input rows must hold nsamp_out + dd_subband_max_shift samples. */
typedef struct dd_subband dd_subband;
int     dd_subband_create(dd_subband** out, int nchans, double fch1, double foff, double tsamp,
                          const double* dm_list, int ndm, int chans_per_subband, int dms_per_nominal);
void    dd_subband_destroy(dd_subband* s);
int64_t dd_subband_max_shift(const dd_subband* s);
/* X: DEVICE [nchans][in_stride]; D: DEVICE [ndm][out_stride], rows in dm_list order */
int     dd_subband_execute(dd_subband* s, const float* X, int64_t in_stride, float* D, int64_t out_stride,
                           int64_t nsamp_out, void* cuda_stream);

/* ---- coherent multi-beam beamformer (ch. 5: eq 5.1, Alg. 2) feeding the dedisperser
 * on the device.  b(f, t, beam) = sum_a W[f][beam][a] * v[f][t][a]; output = detected power |b|^2.
 * V: DEVICE uint8 [nchans][nsamp][nants] (antenna fastest, four antennas per 32-bit word);
 *    each byte: low nibble = real part, high nibble = imaginary part, 4-bit two's complement (-8..7);
 *    nants must be a multiple of 4.
 * W: DEVICE float32 pairs (re, im), [nchans][nbeams][nants]: the weights that point the beams, fixed over
 *    the buffer; no conjugation is applied.
 * P: DEVICE float32 [nbeams][nchans][nsamp] with strides out_stride (channel rows) and out_beam_stride,
 *    i.e. exactly the X layout of dd_execute with nbeams beams.
 * The products run on the tensor cores (fp16 operands -- the 4-bit voltages exactly, the weights as two
 * fp16 terms -- with float32 accumulation): |P - exact| <= 1e-5 (sum_a |W||v|)^2.  Enqueued on cuda_stream. */
int     dd_beamform_power_u4(const uint8_t* V, int nants, int nchans, int64_t nsamp, const float* W, int nbeams,
                             float* P, int64_t out_stride, int64_t out_beam_stride, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* DEDISP_B200_H */
