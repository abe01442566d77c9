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
typedef struct { float re, im; } spiir_c64;

typedef enum {
    SPIIR_OK = 0,
    SPIIR_EINVAL = 1,       /* bad argument; nothing enqueued                                   */
    SPIIR_ENOMEM = 2,       /* host or device allocation failed                                 */
    SPIIR_ECUDA = 3,        /* CUDA runtime error (text in spiir_last_error)                    */
    SPIIR_EUNSUPPORTED = 4, /* shape outside what the kernels are built for                     */
    SPIIR_ESTATE = 5        /* plan used inconsistently (e.g. block longer than max_block)      */
} spiir_status;

/* Options of spiir_plan_create; NULL means {1, 4096, 0, 0}. */
typedef struct {
    int n_streams;     /* S >= 1 independent strain streams sharing the bank (configs[4]: 2)    */
    int max_block;     /* largest n passed to spiir_filter (history / scratch are sized for it) */
    int time_chunks;   /* 0 = choose automatically; 1 = never split a block along time;
                          c > 1 = force the chunked linear scan with c chunks per block         */
    int flags;         /* bit 0: skip the bank-conflict-avoiding filter permutation             */
} spiir_plan_opts;

#define SPIIR_DOWN2 0
#define SPIIR_UP2 1

/* ---------------------------------------------------------------------------------------------
 * Single-rate bank.  PAPER.md:63-67 (Eq. 7, 8); BASELINE.json north_star (1).
 *   a1, b0 : HOST, row-major [n_templates][n_filters] complex64
 *   delays : HOST, row-major [n_templates][n_filters] int32, 0 <= d < 2^20
 *   rate_hz: metadata only (checked by the multirate plan); no arithmetic depends on it
 * Ragged banks are expressed by padding with b0 = 0 filters (reading F6).
 * The plan owns device copies of the re-laid-out coefficients, the filter state
 * y[S][T][L] (zero after create / reset) and the input history (zero after create / reset).
 * ------------------------------------------------------------------------------------------- */
spiir_status spiir_plan_create(spiir_plan_t** out, const spiir_c64* a1, const spiir_c64* b0,
                               const int32_t* delays, int n_templates, int n_filters, int rate_hz,
                               const spiir_plan_opts* opts);

/* One streamed block.  x: DEVICE float32 [S][n]; snr_out: DEVICE complex64 [S][T][n], fully
 * overwritten; 0 <= n <= max_block (n = 0 is a no-op).  State and history advance by n samples. */
spiir_status spiir_filter(spiir_plan_t* p, const float* x, int n, spiir_c64* snr_out, void* cuda_stream);

/* y = 0 and history = 0 (enqueued on the stream). */
spiir_status spiir_plan_reset(spiir_plan_t* p, void* cuda_stream);
void         spiir_plan_destroy(spiir_plan_t* p);

/* Introspection (host side, no GPU work): launch geometry chosen for a block of n samples.
 * Fills: info[0] = filters per lane F, [1] = lanes per template, [2] = warps per CTA,
 * [3] = grid size, [4] = time chunks, [5] = dynamic shared memory bytes, [6] = time tile length,
 * [7] = kernels launched per spiir_filter call. */
spiir_status spiir_plan_launch_info(const spiir_plan_t* p, int n, int info[8]);

/* Copy the carried filter state out / in (DEVICE complex64 [S][T][L], original filter order):
 * the streaming resume state (checkpoint / resume). */
spiir_status spiir_plan_get_state(spiir_plan_t* p, spiir_c64* y_out, void* cuda_stream);
spiir_status spiir_plan_set_state(spiir_plan_t* p, const spiir_c64* y_in, void* cuda_stream);

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
 *   max_block: largest n_in of a call.
 * ------------------------------------------------------------------------------------------- */
spiir_status spiir_resamp_create(spiir_resamp_t** out, int direction, int n_taps, double kaiser_beta,
                                 double cutoff, int n_rows, int max_block);
/* in: DEVICE float32 [rows][n_in], n_in even; out: DEVICE float32 [rows][n_in/2]. */
spiir_status spiir_resample_down(spiir_resamp_t* r, const float* in, int n_in, float* out, void* cuda_stream);
/* in: DEVICE complex64 [rows][n_in]; out: DEVICE complex64 [rows][2*n_in];
 * accumulate != 0: out += up2(in) ("upsampled and added"), else out = up2(in). */
spiir_status spiir_resample_up(spiir_resamp_t* r, const spiir_c64* in, int n_in, spiir_c64* out,
                               int accumulate, void* cuda_stream);
spiir_status spiir_resamp_reset(spiir_resamp_t* r, void* cuda_stream);
void         spiir_resamp_destroy(spiir_resamp_t* r);

/* ---------------------------------------------------------------------------------------------
 * Multirate plan (Fig. 1).  rates_hz descending, each exactly half the previous.
 *   a1[h], b0[h], delays[h]: HOST [n_templates][n_filters_per_rate[h]] for rate h (delays in
 *   samples AT rate h, reading F2).  Options: NULL = {1, rates_hz[0], 192, 5.0, 0.25}.
 * spiir_mr_filter: x DEVICE float32 [S][n] at the base rate, n a multiple of 2^(H-1), n <= max_block;
 * snr_out DEVICE complex64 [S][T][n] at the base rate.  All histories carried across calls.
 * ------------------------------------------------------------------------------------------- */
typedef struct {
    int n_streams;
    int max_block;       /* at the base rate */
    int n_taps;          /* 192 (BASELINE.json configs[3]) */
    double kaiser_beta;  /* 5.0 */
    double cutoff;       /* 0.25 cycles per high-rate sample */
} spiir_mr_opts;

spiir_status spiir_mr_plan_create(spiir_mr_plan_t** out, int n_rates, const int* rates_hz,
                                  const spiir_c64* const* a1, const spiir_c64* const* b0,
                                  const int32_t* const* delays, const int* n_filters_per_rate,
                                  int n_templates, const spiir_mr_opts* opts);
spiir_status spiir_mr_filter(spiir_mr_plan_t* p, const float* x, int n, spiir_c64* snr_out, void* cuda_stream);
spiir_status spiir_mr_plan_reset(spiir_mr_plan_t* p, void* cuda_stream);
void         spiir_mr_plan_destroy(spiir_mr_plan_t* p);
/* Number of kernels one spiir_mr_filter call of n base-rate samples launches. */
int          spiir_mr_launches(const spiir_mr_plan_t* p, int n);

/* ---------------------------------------------------------------------------------------------
 * Host-only helpers (no GPU work; usable without a CUDA device): the plan's filter permutation
 * and launch geometry, exposed so that they can be inspected and tested.
 *   spiir_host_layout: pos_out [T*L] = index of filter (t, l) in the plan's [G][F][32] arrays;
 *     coef_out [G*F*32*4], dly_out [G*F*32] (any may be NULL); info = {F, lanes per template, G,
 *     G*F*32}; conflict_degree = mean over quarter-warp window reads of the worst 16-byte
 *     bank-group multiplicity (1.0 = conflict free).
 *   spiir_host_geometry: info as spiir_plan_launch_info, for a device with n_sm SMs and
 *     smem_optin bytes of opt-in shared memory per block.
 * ------------------------------------------------------------------------------------------- */
spiir_status spiir_host_layout(const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays, int n_templates,
                               int n_filters, int avoid_conflicts, int32_t* pos_out, float* coef_out,
                               int32_t* dly_out, int info[4], double* conflict_degree);
spiir_status spiir_host_geometry(int n_templates, int n_filters, int n_streams, int max_delay, int n,
                                 int time_chunks, int n_sm, int smem_optin, int info[8]);

/* Measurement aid (not part of the hot path): times a register-only FFMA loop on the current device and
 * returns the FP32 rate it reached in TFLOP/s (2 flop per FMA).  Synchronises the device.  bench.py reports
 * the ALU roofline against the nominal peak (SMs x 128 lanes x 2 x clock) and quotes this number beside it
 * ("achieved FP32 peak"). */
spiir_status spiir_probe_fp32_peak(double* tflops_out);

const char*  spiir_last_error(void);
/* "spiir-b200 <version> sm_100a" */
const char*  spiir_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPIIR_H */
