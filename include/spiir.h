/*
 * spiir.h -- C ABI of the B200-native SPIIR hot path (arXiv:1702.02256).
 *
 * Citations are lines of /root/reference/PAPER.md ("PAPER.md:<line>") plus the readings listed
 * in DESIGN.md (F1..F10, R1..R9).
 *
 * WHAT IS COMPUTED
 *   Single-rate bank (Eq. 7 and Eq. 8):
 *       y_l[k] = a1_l * y_l[k-1] + b0_l * x[k - d_l]          (complex one-pole filter, real input)
 *       z[k]   = sum_l y_l[k]                                  (complex SNR series of one template)
 *   for T templates of L filters each against S float32 strain streams.  The factor 2*dt of
 *   Eq. 8 is folded into b0 by the caller (reading F1).  Delays are integer samples at the rate
 *   the bank runs at (F2); d = 0 is allowed (F3); x[k] = 0 for k < 0 and y[-1] = 0 (F4).
 *   Consecutive spiir_filter calls continue ONE stream: filter state y and the last d_max input
 *   samples are carried, so any partition into blocks equals one long call.
 *
 *   Resampling (Eq. 9; readings R1-R3): one N-tap Kaiser-windowed-sinc low pass
 *       h[j] = g * I0(beta*sqrt(1-(2j/(N-1)-1)^2))/I0(beta) * 2fc * sinc(2fc*(j-(N-1)/2)),  sum h = 1
 *   applied causally with zero pre-history:
 *       down-by-2:  v[m]    = sum_{j<N}   h[j]    * u[2m-j]
 *       up-by-2:    w[2m+p] = 2 * sum_{q<N/2} h[2q+p] * v[m-q],  p in {0,1}   (complex rows)
 *
 *   Multirate (Fig. 1; R4-R7): x_0 = x, x_h = down2(x_{h-1}); z_h = bank_h(x_h);
 *   acc_{H-1} = z_{H-1}; acc_{h-1} = z_{h-1} + up2(acc_h); result acc_0 at the base rate.
 *
 * CONVENTIONS
 *   - spiir_c64 is interleaved (re, im) float32 == numpy/torch complex64 == CUDA float2.
 *   - "host" pointers are read during the call and may be freed afterwards; "device" pointers
 *     are CUDA device memory owned by the caller (e.g. torch tensors) and must stay valid until
 *     the work enqueued on the stream has finished.
 *   - DEVICE MEMORY: every create call takes an optional caller-owned device workspace in its
 *     options struct (size from the matching *_workspace_bytes call, 256-byte aligned, lent to the
 *     plan for its lifetime; the Python binding passes one torch tensor).  With a workspace the
 *     library makes no cudaMalloc at all; with workspace == NULL it allocates one block itself.
 *     Compute calls never allocate.
 *   - Every compute call only ENQUEUES work on `cuda_stream` (a cudaStream_t passed as void*,
 *     NULL = default stream) and returns without synchronising.  A plan may be used from one
 *     stream at a time; plans are not thread-safe.
 *   - Errors: argument errors return SPIIR_EINVAL and enqueue nothing; CUDA failures return
 *     SPIIR_ECUDA / SPIIR_ENOMEM.  spiir_last_error() gives a thread-local message.
 *   - A compute call enqueues the SAME kernels with the SAME arguments for every block of a stream
 *     (which half of each ping-pong history is current is a word in device memory, flipped by the
 *     kernels themselves), so one call captured into a CUDA graph can be replayed for every block
 *     as long as x / snr_out / n stay the same.  The multirate call forks onto plan-owned side
 *     streams with events and joins before it returns control of `cuda_stream` (capturable).
 *   - There is no CPU fallback: without a CUDA device every create call fails with SPIIR_ECUDA.
 *   - Arithmetic is IEEE float32 with FMA contraction; the sum over filters is taken in a fixed,
 *     plan-determined order (deterministic, reading F8).
 */
#ifndef SPIIR_H
#define SPIIR_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct spiir_plan    spiir_plan_t;    /* single-rate bank + its streaming state       */
typedef struct spiir_resamp  spiir_resamp_t;  /* one x2 stage: taps + FIR history              */
typedef struct spiir_mr_plan spiir_mr_plan_t; /* multirate: H banks + (H-1) down + (H-1) up    */
typedef struct spiir_pd_plan spiir_pd_plan_t; /* the paper's own (Maxwell) kernel design, for comparison */
typedef struct { float re, im; } spiir_c64;

typedef enum {
    SPIIR_OK = 0,
    SPIIR_EINVAL = 1,       /* bad argument; nothing enqueued                                   */
    SPIIR_ENOMEM = 2,       /* host or device allocation failed / workspace too small           */
    SPIIR_ECUDA = 3,        /* CUDA runtime error (text in spiir_last_error)                    */
    SPIIR_EUNSUPPORTED = 4, /* shape outside what the kernels are built for                     */
    SPIIR_ESTATE = 5        /* plan used inconsistently (e.g. block longer than max_block)      */
} spiir_status;

/* Options of spiir_plan_create / spiir_plan_create_ragged; NULL means {1, 4096, 0, 0, NULL, 0}. */
typedef struct {
    int n_streams;     /* S >= 1 independent strain streams sharing the bank (configs[4]: 2)    */
    int max_block;     /* largest n passed to spiir_filter (history / scratch are sized for it) */
    int time_chunks;   /* 0 = choose automatically; 1 = never split a block along time;
                          c > 1 = force the chunked linear scan with c chunks per block         */
    int flags;         /* bit 0: skip the bank-conflict-avoiding filter permutation             */
    void*  workspace;        /* DEVICE, caller-owned, 256-byte aligned; NULL: the library allocates */
    size_t workspace_bytes;  /* >= the matching spiir_plan_workspace_bytes[_ragged] value        */
} spiir_plan_opts;

#define SPIIR_DOWN2 0
#define SPIIR_UP2 1

/* ---------------------------------------------------------------------------------------------
 * Single-rate bank.  PAPER.md:63-67 (Eq. 7, 8); BASELINE.json north_star (1).
 *   a1, b0 : HOST, row-major [n_templates][n_filters] complex64
 *   delays : HOST, row-major [n_templates][n_filters] int32, 0 <= d < 2^20
 *   rate_hz: metadata only (checked by the multirate plan); no arithmetic depends on it
 *   n_filters: 1 .. 2048.  Up to 512 filters a template is one warp (or part of one); beyond that
 *   it spans several warps of one CTA ("513 filters -> 544 threads").
 * The plan owns device copies of the re-laid-out coefficients, the filter state
 * y[S][T][L] (zero after create / reset) and the input history (zero after create / reset).
 *
 * spiir_plan_workspace_bytes: device bytes spiir_plan_create needs for this shape on the current
 * device (0 on error); max_delay = the largest delay of the bank; time_chunks as in the options.
 * ------------------------------------------------------------------------------------------- */
size_t       spiir_plan_workspace_bytes(int n_templates, int n_filters, int max_delay, int n_streams,
                                        int max_block, int time_chunks);
spiir_status spiir_plan_create(spiir_plan_t** out, const spiir_c64* a1, const spiir_c64* b0,
                               const int32_t* delays, int n_templates, int n_filters, int rate_hz,
                               const spiir_plan_opts* opts);

/* Ragged bank: template t owns filters [filter_offsets[t], filter_offsets[t+1]) of the flat HOST
 * arrays a1, b0, delays (CSR layout; filter_offsets HOST int32 [n_templates + 1], non-decreasing,
 * every template 1 .. 2048 filters).  PAPER.md:102-112 ("a template with 513 filters ... a template
 * with 5 filters ...; four small templates in a single warp"), PAPER.md:275 (zero padding is the
 * paper's own workaround).  Templates are grouped into classes of equal lane mapping; inside a
 * class each template is padded only up to its warp tile (the paper's "not more than 31 idle
 * threads" per warp row), never to the longest template of the bank.  snr_out keeps the caller's
 * template order.  State order of get/set_state: flat CSR order. */
size_t       spiir_plan_workspace_bytes_ragged(const int32_t* filter_offsets, int n_templates, int max_delay,
                                               int n_streams, int max_block, int time_chunks);
spiir_status spiir_plan_create_ragged(spiir_plan_t** out, const spiir_c64* a1, const spiir_c64* b0,
                                      const int32_t* delays, const int32_t* filter_offsets, int n_templates,
                                      int rate_hz, const spiir_plan_opts* opts);

/* One streamed block.  x: DEVICE float32 [S][n]; snr_out: DEVICE complex64 [S][T][n], fully
 * overwritten; 0 <= n <= max_block (n = 0 is a no-op).  State and history advance by n samples. */
spiir_status spiir_filter(spiir_plan_t* p, const float* x, int n, spiir_c64* snr_out, void* cuda_stream);

/* y = 0 and history = 0 (enqueued on the stream). */
spiir_status spiir_plan_reset(spiir_plan_t* p, void* cuda_stream);
void         spiir_plan_destroy(spiir_plan_t* p);

/* Introspection (host side, no GPU work): launch geometry chosen for a block of n samples (for a ragged
 * plan: of its largest class).  Fills: info[0] = filters per lane F, [1] = lanes per template,
 * [2] = warps per CTA, [3] = grid size, [4] = time chunks, [5] = dynamic shared memory bytes,
 * [6] = time tile length, [7] = kernels launched per spiir_filter call (all classes). */
spiir_status spiir_plan_launch_info(const spiir_plan_t* p, int n, int info[8]);

/* The streaming resume state (checkpoint / resume): BOTH the filter state y
 * (DEVICE complex64 [S][T][L], original filter order; ragged: [S][total filters] in CSR order) AND
 * the input history (DEVICE float32 [S][spiir_plan_history_len], oldest sample first = the last
 * max_delay samples of the stream; may be NULL when the length is 0).  A fresh plan of the same
 * bank after set_state continues the stream exactly as the original plan would have. */
int          spiir_plan_history_len(const spiir_plan_t* p);
spiir_status spiir_plan_get_state(spiir_plan_t* p, spiir_c64* y_out, float* hist_out, void* cuda_stream);
spiir_status spiir_plan_set_state(spiir_plan_t* p, const spiir_c64* y_in, const float* hist_in, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Kaiser-windowed-sinc taps (Eq. 9; readings R1-R3), computed in double and
 * rounded once to float32.  taps_out: HOST float32 [n_taps].
 * ------------------------------------------------------------------------------------------- */
spiir_status spiir_kaiser_taps(int n_taps, double kaiser_beta, double cutoff, float* taps_out);

/* ---------------------------------------------------------------------------------------------
 * One streaming x2 resampling stage over n_rows independent rows.
 *   direction SPIIR_DOWN2: rows are real float32;   history = n_taps-1 samples per row
 *   direction SPIIR_UP2  : rows are complex64;      history = n_taps/2-1 samples per row
 *   n_taps even, 2 <= n_taps <= 1024; taps are spiir_kaiser_taps(n_taps, kaiser_beta, cutoff).
 *   Register-blocked kernels exist for 384 / 192 / 32 taps (the paper's 384-tap
 *   down and 32-tap up filters; configs[3]: 192), a generic kernel serves every other count.
 *   The 192-tap and the 32-tap up stage of a large call (rows * n_in >= 65536) run on the tensor cores: the polyphase FIR as
 *   a banded-Toeplitz contraction, tcgen05 kind::tf32 with every operand split into a TF32-exact high part and
 *   its float32 remainder; the product of the high parts and two bf16 correction products accumulate in TMEM
 *   (rel-L2 8.5e-7 against the float64 oracle).  The input is fetched through a tensor map that is
 *   encoded on the host in every call (needs cuTensorMapEncodeTiled from the installed driver, no libcuda link).
 *   opts: NULL means {4096, NULL, 0, 0}.
 * ------------------------------------------------------------------------------------------- */
typedef struct {
    int    max_block;        /* largest n_in of a call */
    void*  workspace;        /* DEVICE, caller-owned; NULL: the library allocates */
    size_t workspace_bytes;
    int    flags;            /* bit 0: never use the tensor-core kernel (192 / 32-tap up stage), for A/B measurements */
} spiir_resamp_opts;

size_t       spiir_resamp_workspace_bytes(int direction, int n_taps, int n_rows);
spiir_status spiir_resamp_create(spiir_resamp_t** out, int direction, int n_taps, double kaiser_beta,
                                 double cutoff, int n_rows, const spiir_resamp_opts* opts);
/* in: DEVICE float32 [rows][n_in], n_in even; out: DEVICE float32 [rows][n_in/2]. */
spiir_status spiir_resample_down(spiir_resamp_t* r, const float* in, int n_in, float* out, void* cuda_stream);
/* in: DEVICE complex64 [rows][n_in] (8-byte aligned); out: DEVICE complex64 [rows][2*n_in] (16-byte aligned);
 * accumulate != 0: out += up2(in) ("upsampled and added"), else out = up2(in). */
spiir_status spiir_resample_up(spiir_resamp_t* r, const spiir_c64* in, int n_in, spiir_c64* out,
                               int accumulate, void* cuda_stream);
spiir_status spiir_resamp_reset(spiir_resamp_t* r, void* cuda_stream);
void         spiir_resamp_destroy(spiir_resamp_t* r);
/* Resume state of a stage: its input history, DEVICE [rows][spiir_resamp_history_len] (float32 for a
 * down stage, complex64 for an up stage), oldest first. */
int          spiir_resamp_history_len(const spiir_resamp_t* r);
spiir_status spiir_resamp_get_state(spiir_resamp_t* r, void* hist_out, void* cuda_stream);
spiir_status spiir_resamp_set_state(spiir_resamp_t* r, const void* hist_in, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Multirate plan (Fig. 1).  rates_hz descending, each exactly half the previous.
 *   a1[h], b0[h], delays[h]: HOST [n_templates][n_filters_per_rate[h]] for rate h (delays in
 *   samples AT rate h, reading F2).
 *   Options: separate down / up filters (~100 dB / 384 taps down, ~60 dB / 32 taps
 *   up); NULL = {1, rates_hz[0], 192, 5.0, 0.25, 192, 5.0, 0.25, NULL, 0} (BASELINE.json configs[3]).
 * spiir_mr_filter: x DEVICE float32 [S][n] at the base rate, n a multiple of 2^(H-1), n <= max_block;
 * snr_out DEVICE complex64 [S][T][n] at the base rate (16-byte aligned).  All histories carried.
 * ------------------------------------------------------------------------------------------- */
typedef struct {
    int n_streams;
    int max_block;            /* at the base rate */
    int n_taps_down;  double kaiser_beta_down;  double cutoff_down;   /* 192, 5.0, 0.25 cycles per high-rate sample */
    int n_taps_up;    double kaiser_beta_up;    double cutoff_up;
    void*  workspace;         /* DEVICE, caller-owned; NULL: the library allocates */
    size_t workspace_bytes;
} spiir_mr_opts;

/* max_delay_per_rate: HOST int [n_rates], the largest delay of each rate's bank. */
size_t       spiir_mr_workspace_bytes(int n_rates, const int* n_filters_per_rate, const int* max_delay_per_rate,
                                      int n_templates, const spiir_mr_opts* opts);
spiir_status spiir_mr_plan_create(spiir_mr_plan_t** out, int n_rates, const int* rates_hz,
                                  const spiir_c64* const* a1, const spiir_c64* const* b0,
                                  const int32_t* const* delays, const int* n_filters_per_rate,
                                  int n_templates, const spiir_mr_opts* opts);
spiir_status spiir_mr_filter(spiir_mr_plan_t* p, const float* x, int n, spiir_c64* snr_out, void* cuda_stream);
spiir_status spiir_mr_plan_reset(spiir_mr_plan_t* p, void* cuda_stream);
void         spiir_mr_plan_destroy(spiir_mr_plan_t* p);
/* Number of kernels one spiir_mr_filter call of n base-rate samples launches. */
int          spiir_mr_launches(const spiir_mr_plan_t* p, int n);
/* Resume state as one DEVICE blob of spiir_mr_plan_state_bytes bytes: for every rate h (highest first) the
 * bank's y [S][T][L_h] complex64 then its input history [S][max_delay_h] float32; then the histories of the
 * down stages (rate 0->1 first), then those of the up stages (1->0 first); each section 16-byte aligned. */
size_t       spiir_mr_plan_state_bytes(const spiir_mr_plan_t* p);
spiir_status spiir_mr_plan_get_state(spiir_mr_plan_t* p, void* blob_out, void* cuda_stream);
spiir_status spiir_mr_plan_set_state(spiir_mr_plan_t* p, const void* blob_in, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Rate assignment: "the a1 coefficient determines the upper bound of the frequency band
 * of the filter, and thus the Nyquist rate ...; we round the Nyquist rate of the filter to the nearest
 * biggest available rate".  The paper gives no formula; reading R8: a1 = |a1| e^{i w} is a damped
 * complex exponential with centre frequency f0 = |w| R / (2 pi) and half-power half-width
 * df = -ln|a1| R / (2 pi); its band upper bound is f_hi = f0 + band_factor * df, its Nyquist rate 2 f_hi,
 * and it is assigned to the LOWEST available rate >= 2 f_hi (the base rate if none is).
 *   a1 HOST complex64 [n] at rate base_rate_hz; rates_hz HOST int [n_rates] descending, rates_hz[0] ==
 *   base_rate_hz; rate_index_out HOST int32 [n].  Host only, off the hot path.
 * ------------------------------------------------------------------------------------------- */
spiir_status spiir_assign_rates(const spiir_c64* a1, int n, int base_rate_hz, const int* rates_hz, int n_rates,
                                double band_factor, int32_t* rate_index_out);

/* ---------------------------------------------------------------------------------------------
 * Host-only helpers (no GPU work; usable without a CUDA device): the plan's filter permutation
 * and launch geometry, exposed so that they can be inspected and tested.
 *   spiir_host_layout: pos_out [T*L] = index of filter (t, l) in the plan's [G][F][32] arrays;
 *     coef_out [G*F*32*4], dly_out [G*F*32] (any may be NULL); info = {F, lanes per template, G,
 *     G*F*32}; conflict_degree = mean over quarter-warp window reads of the worst 16-byte
 *     bank-group multiplicity (1.0 = conflict free).
 *   spiir_host_geometry: info as spiir_plan_launch_info, for a device with n_sm SMs and
 *     smem_optin bytes of opt-in shared memory per block.
 *   spiir_host_lane_mapping: info = {F, lanes per template, warps per template} for L filters per template
 *     in a bank of T templates.
 * ------------------------------------------------------------------------------------------- */
spiir_status spiir_host_layout(const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays, int n_templates,
                               int n_filters, int avoid_conflicts, int32_t* pos_out, float* coef_out,
                               int32_t* dly_out, int info[4], double* conflict_degree);
spiir_status spiir_host_geometry(int n_templates, int n_filters, int n_streams, int max_delay, int n,
                                 int time_chunks, int n_sm, int smem_optin, int info[8]);
spiir_status spiir_host_lane_mapping(int n_filters, int n_templates, int info[3]);

/* ---------------------------------------------------------------------------------------------
 * NO-ALLOCATION ENTRY POINT (Eq. 7-8; the time-parallel scan of SURVEY.md section 8 row a7).
 * For callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that
 * forbid it): filters ONE block from zero state (y = 0, x[k] = 0 for k < 0) with no plan and no workspace.
 *   a1, b0   : DEVICE [n_templates][n_filters] complex64, caller order (not permuted)
 *   delays   : DEVICE [n_templates][n_filters] int32, >= 0
 *   x        : DEVICE [n] float32;   snr_out : DEVICE [n_templates][n] complex64, overwritten
 *   time_chunks : 0 = as many chunks of >= 64 samples as fit (at most 64), else that many chunks
 * The chunk states of the scan (n_templates * n_filters * chunks * 8 bytes, spiir_noalloc_scratch_need) live in a
 * device array built into the library: SPIIR_NOALLOC_SCRATCH_BYTES (4 MiB) on every GPU that loads the library,
 * held until the process exits.  A call that needs more returns SPIIR_EINVAL with a message and launches nothing;
 * n_filters > 512 returns SPIIR_EUNSUPPORTED.  The call makes no cudaMalloc / cudaFree / allocating library call
 * and does not synchronise; three kernels are enqueued on cuda_stream.  spiir_noalloc_setup looks the array's
 * device address up for the current device (done lazily by the first call otherwise; call it once before a stream
 * capture).  All calls share the array: calls on ONE stream are ordered and safe, calls that overlap on the GPU
 * (several streams, concurrent graph replays) RACE.  Nothing in the array needs clearing between calls (every word
 * a call reads it has written itself).  Results agree with spiir_filter on a fresh plan within the parity tolerance
 * (float32, another summation order); deterministic.  Owns nothing, keeps no state between calls.
 * ------------------------------------------------------------------------------------------- */
#define SPIIR_NOALLOC_SCRATCH_BYTES (4u << 20)
size_t       spiir_noalloc_scratch_need(int n_templates, int n_filters, int n, int time_chunks);
spiir_status spiir_noalloc_setup(void);
spiir_status spiir_filter_block_noalloc(const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays, int n_templates,
                                        int n_filters, const float* x, int n, int time_chunks, spiir_c64* snr_out,
                                        void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * COMPARISON KERNELS, not the product path: the paper's own single-rate design restated
 * for the same B200 so that the new mapping can be measured against it on one machine (bench.py --impl
 * paper_design).  One thread per filter; a template of more than 32 filters is one CUDA block of
 * ceil(L/32)*32 threads ("block-based kernel"), templates of <= 32 filters take next_pow2(L) threads and share
 * warps, 256 threads per block ("warp-based kernel"); coefficients by coalesced global loads, y in a register,
 * x through the read-only data cache (__ldg), per-sample warp-shuffle sum, warp partials combined with
 * atomicAdd into the global SNR ("DA").  Same streaming semantics and layouts as spiir_filter
 * (snr_out is zero-filled, then accumulated).  Float atomics: the summation order is not fixed (reading F8).
 * ------------------------------------------------------------------------------------------- */
spiir_status spiir_pd_plan_create(spiir_pd_plan_t** out, const spiir_c64* a1, const spiir_c64* b0,
                                  const int32_t* delays, int n_templates, int n_filters, int max_block);
spiir_status spiir_pd_filter(spiir_pd_plan_t* p, const float* x, int n, spiir_c64* snr_out, void* cuda_stream);
spiir_status spiir_pd_plan_reset(spiir_pd_plan_t* p, void* cuda_stream);
void         spiir_pd_plan_destroy(spiir_pd_plan_t* p);

/* ---------------------------------------------------------------------------------------------
 * MEASUREMENT AIDS for bench.py, not part of the product surface (they allocate, run for milliseconds and
 * synchronise the device).
 *   spiir_probe_fp32_peak: TFLOP/s of a register-only FFMA loop with shared constant operands (the nominal
 *     FP32 rate: 2 flop per lane per clock).
 *   spiir_probe_ffma2_operands: cycles per packed FFMA2 warp-instruction on one SM sub-partition when the
 *     instruction reads 3, 4, 5 and 6 distinct 32-bit register words (4 warps per sub-partition).  The Eq. 7
 *     update needs two 5-word FFMA2s per filter-sample; DESIGN.md 5.1 derives the kernel's ceiling from it.
 * ------------------------------------------------------------------------------------------- */
spiir_status spiir_probe_fp32_peak(double* tflops_out);
spiir_status spiir_probe_ffma2_operands(double cycles_out[4]);

const char*  spiir_last_error(void);
/* "spiir-b200 <version> sm_100a" */
const char*  spiir_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPIIR_H */
