// spiir_resample.cuh -- sm_100a kernels for the x2 polyphase FIR stages of the multirate scheme
// (Eq. 9).
//
//   down-by-2 (real rows):    v[m]    = sum_{j<N}    h[j]    * u[2m - j]
//   up-by-2   (complex rows): w[2m+p] = 2 * sum_{q<N/2} h[2q+p] * v[m - q],   p in {0, 1}
//
// Both keep the row history (N-1 real / N/2-1 complex samples) across calls in a ping-pong pair:
// a call reads hist + in and the CTA that owns the first tile of a row writes hist_next.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "spiir_common.cuh"   // phase_read / last_cta_arrives

namespace spiir {

constexpr int kMaxTaps = 1024;

struct ResampArgs {
    const float* taps;      // [N] float32 taps (device)
    const void*  in;        // down: float [rows][n_in]; up: float2 [rows][n_in]
    void*        out;       // down: float [rows][n_in/2]; up: float2 [rows][2 n_in]
    void*        hbuf[2];   // down: float [rows][N-1]; up: float2 [rows][N/2-1]; ping-pong, hbuf[phase] is current
    int*         phase;     // device words {phase, arrivals} (see spiir_filter.cuh)
    int rows, n_in, N;
    int tile;               // down: outputs per CTA; up: inputs per CTA
    int accumulate;         // up only
};

// ---------------------------------------------------------------------------------------------
// Down-by-2.  grid = (rows, tiles), block = 128 threads.  Shared: taps[N], even/odd input phases
// so that lanes read consecutive words: u[2m-2q] = ue[m-q], u[2m-2q-1] = uo[m-q-1].
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) spiir_down2_kernel(const ResampArgs a)
{
    extern __shared__ __align__(16) float sm[];
    const int N = a.N, H = N - 1, half = N / 2;
    const int row = blockIdx.x, m0 = blockIdx.y * a.tile;
    const int n_out = a.n_in >> 1;
    const int tm = min(a.tile, n_out - m0);
    float* taps = sm;                               // [N]
    float* ue = taps + N;                           // ue[i] = u[2(m0 - half + i)],     i in [0, tm+half)
    float* uo = ue + (a.tile + half);               // uo[i] = u[2(m0 - half + i) + 1]
    const int ph = phase_read(a.phase);
    const float* in = reinterpret_cast<const float*>(a.in) + (size_t)row * a.n_in;
    const float* hist = reinterpret_cast<const float*>(a.hbuf[ph]) + (size_t)row * H;
    for (int i = threadIdx.x; i < N; i += blockDim.x) taps[i] = a.taps[i];
    const int base = 2 * (m0 - half);               // first input sample staged (may be < 0 -> history)
    for (int i = threadIdx.x; i < 2 * (tm + half); i += blockDim.x) {
        const int g = base + i;                     // sample index relative to the block start
        float v = 0.f;
        if (g >= 0) v = in[g];
        else if (H + g >= 0) v = hist[H + g];
        if (i & 1) uo[i >> 1] = v; else ue[i >> 1] = v;
    }
    __syncthreads();
    for (int ml = threadIdx.x; ml < tm; ml += blockDim.x) {
        // v[m] = sum_q h[2q] ue[m-q] + h[2q+1] uo[m-q-1];  local index of m is ml + half
        float acc0 = 0.f, acc1 = 0.f;
        const int c = ml + half;
#pragma unroll 8
        for (int q = 0; q < half; ++q) {
            acc0 = fmaf(taps[2 * q], ue[c - q], acc0);
            acc1 = fmaf(taps[2 * q + 1], uo[c - q - 1], acc1);
        }
        reinterpret_cast<float*>(a.out)[(size_t)row * n_out + m0 + ml] = acc0 + acc1;
    }
    if (blockIdx.y == 0 && H > 0) {                 // carried history: last H samples of hist ++ in
        float* hn = reinterpret_cast<float*>(a.hbuf[ph ^ 1]) + (size_t)row * H;
        for (int i = threadIdx.x; i < H; i += blockDim.x) {
            const int g = a.n_in - H + i;
            hn[i] = (g >= 0) ? in[g] : hist[a.n_in + i];
        }
    }
    if (last_cta_arrives(a.phase, gridDim.x * gridDim.y)) a.phase[0] = ph ^ 1;
}

// ---------------------------------------------------------------------------------------------
// Up-by-2 (+ accumulate).  grid = (rows, tiles), block = 128 threads; one thread per input sample
// m produces w[2m] and w[2m+1] with (re, im) packed FMAs.  Shared: taps[N] split by phase, the
// input segment v[m0-(N/2-1) .. m0+tile).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) spiir_up2_kernel(const ResampArgs a)
{
    extern __shared__ __align__(16) float sm[];
    const int N = a.N, half = N / 2, H = half - 1;
    const int row = blockIdx.x, m0 = blockIdx.y * a.tile;
    const int tm = min(a.tile, a.n_in - m0);
    float* tp0 = sm;                                // h[2q]
    float* tp1 = sm + half;                         // h[2q+1]
    float2* vs = reinterpret_cast<float2*>(sm + N); // vs[i] = v[m0 - H + i], i in [0, tm+H)
    const int ph = phase_read(a.phase);
    const float2* in = reinterpret_cast<const float2*>(a.in) + (size_t)row * a.n_in;
    const float2* hist = reinterpret_cast<const float2*>(a.hbuf[ph]) + (size_t)row * H;
    for (int i = threadIdx.x; i < half; i += blockDim.x) { tp0[i] = a.taps[2 * i]; tp1[i] = a.taps[2 * i + 1]; }
    for (int i = threadIdx.x; i < tm + H; i += blockDim.x) {
        const int g = m0 - H + i;
        float2 v = make_float2(0.f, 0.f);
        if (g >= 0) v = in[g];
        else if (H + g >= 0) v = hist[H + g];
        vs[i] = v;
    }
    __syncthreads();
    float2* out = reinterpret_cast<float2*>(a.out) + (size_t)row * 2 * a.n_in;
    for (int ml = threadIdx.x; ml < tm; ml += blockDim.x) {
        float2 acc0 = make_float2(0.f, 0.f), acc1 = make_float2(0.f, 0.f);
        const int c = ml + H;
#pragma unroll 8
        for (int q = 0; q < half; ++q) {
            const float2 v = vs[c - q];
            acc0 = __ffma2_rn(make_float2(tp0[q], tp0[q]), v, acc0);
            acc1 = __ffma2_rn(make_float2(tp1[q], tp1[q]), v, acc1);
        }
        float4 w = make_float4(2.f * acc0.x, 2.f * acc0.y, 2.f * acc1.x, 2.f * acc1.y);
        float4* o = reinterpret_cast<float4*>(out + 2 * (size_t)(m0 + ml));   // 16-byte aligned: even complex index
        if (a.accumulate) { float4 p = *o; w.x += p.x; w.y += p.y; w.z += p.z; w.w += p.w; }
        *o = w;
    }
    if (blockIdx.y == 0 && H > 0) {
        float2* hn = reinterpret_cast<float2*>(a.hbuf[ph ^ 1]) + (size_t)row * H;
        for (int i = threadIdx.x; i < H; i += blockDim.x) {
            const int g = a.n_in - H + i;
            hn[i] = (g >= 0) ? in[g] : hist[a.n_in + i];
        }
    }
    if (last_cta_arrives(a.phase, gridDim.x * gridDim.y)) a.phase[0] = ph ^ 1;
}

// ---------------------------------------------------------------------------------------------
// Register-blocked up-by-2 (+ accumulate) for a compile-time tap count N = 2*HALF.
//
// The generic kernel above issues three shared-memory loads per two packed FMAs and is bound by the
// LSU.  Here a thread owns R = 5 consecutive input positions m0..m0+4, i.e. 10 complex outputs in
// 20 FP32 accumulators, and walks the R + HALF - 1 inputs they depend on once: one 8-byte LDS per
// input feeds up to 4R FFMAs.  The taps are kernel parameters, so they live in constant bank 0 and
// reach the FFMAs through uniform registers (LDCU), not through the vector register file or the LSU;
// the loop is fully unrolled, which makes every tap index a compile-time constant and drops the
// out-of-range (position, tap) pairs.
// R = 5 is odd on purpose: lane l reads smem word pair 5l + const, and 5 is coprime with the 16
// 8-byte banks, so the LDS.64 are conflict free.  Outputs go through shared memory to be written
// (and, for accumulate, read) as coalesced 16-byte accesses.
//
// Work split: a CTA of 128 threads handles `rpc` rows x one segment of `seg` <= 640 inputs, one thread
// per (row, 5 inputs); rpc = 128 / ceil(seg / 5) rows when the rows are short, else 1.  Small CTAs (16 KB
// of shared memory, 48 registers) keep ~10 of them on an SM, so the load / FIR / store phases of
// different CTAs overlap; a persistent double-buffered (cp.async) variant measured slower.
// ---------------------------------------------------------------------------------------------
constexpr int kUpR = 5;

template <int HALF>
struct UpTaps { float t0[HALF]; float t1[HALF]; };    // t0[q] = h[2q], t1[q] = h[2q+1]

constexpr int kUpSegMax = 128 * kUpR;

struct UpArgs {
    const float2* in;        // [rows][n_in]
    float2*       out;       // [rows][2 n_in]
    float2*       hbuf[2];   // [rows][HALF-1] ping-pong, hbuf[phase] is current
    int*          phase;
    int rows, n_in;
    int seg;                 // inputs per row segment (<= kUpSegMax)
    int nseg;                // segments per row
    int upr;                 // units (threads) per row segment = ceil(seg / R)
    int rpc;                 // rows per CTA
    int accumulate;
};

template <int HALF>
__global__ void __launch_bounds__(128, 8) spiir_up2_fir_kernel(const UpArgs a, const __grid_constant__ UpTaps<HALF> taps)
{
    constexpr int R = kUpR, H = HALF - 1;
    extern __shared__ __align__(16) float2 smu[];
    // per row slot: input segment with history [seg + H] (+ pad), then the output tile [2*seg]
    const int in_stride = (a.seg + H + R + 3) & ~1;                     // complex words, even
    const int out_stride = 2 * (a.seg + R);
    float2* vin = smu;                                                  // [rpc][in_stride]
    float2* vout = smu + (size_t)a.rpc * in_stride;                     // [rpc][out_stride]
    const int seg_idx = blockIdx.x % a.nseg;
    const int row0 = (blockIdx.x / a.nseg) * a.rpc;
    const int m_base = seg_idx * a.seg;
    const int seg_len = min(a.seg, a.n_in - m_base);
    const int nrow = min(a.rpc, a.rows - row0);
    const int ph = phase_read(a.phase);
    const float2* hcur = a.hbuf[ph];
    float2* hnext = a.hbuf[ph ^ 1];

    // Short filters (32 taps) are HBM-bound: the tile of `out` that is accumulated into is then fetched with
    // cp.async while the inputs are staged and the FIR runs, and added in shared memory (PREFETCH).  With
    // 192 taps the FIR hides that read anyway and the extra pass only costs issue slots.
    constexpr bool PREFETCH = HALF <= 16;
    const bool pre = PREFETCH && a.accumulate != 0;
    if (pre) {
        for (int sl = 0; sl < nrow; ++sl) {
            const float2* src = a.out + (size_t)(row0 + sl) * 2 * a.n_in + 2 * m_base;
            float2* dst = vout + (size_t)sl * out_stride;
            for (int i = threadIdx.x; i < seg_len; i += blockDim.x) {
                const uint32_t d = (uint32_t)__cvta_generic_to_shared(dst + 2 * i);
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(src + 2 * i) : "memory");
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    // stage inputs: vin[slot][i] = v[row][m_base - H + i], i in [0, seg_len + H); zero beyond
#pragma unroll 4
    for (int sl = 0; sl < nrow; ++sl) {
        const float2* in = a.in + (size_t)(row0 + sl) * a.n_in;
        const float2* hist = hcur + (size_t)(row0 + sl) * H;
        float2* dst = vin + (size_t)sl * in_stride;
        for (int i = threadIdx.x; i < in_stride; i += blockDim.x) {
            const int g = m_base - H + i;
            float2 v = make_float2(0.f, 0.f);
            if (i < seg_len + H) {
                if (g >= 0) v = in[g];
                else if (H + g >= 0) v = hist[H + g];
            }
            dst[i] = v;
        }
    }
    __syncthreads();

    const int slot = threadIdx.x / a.upr, unit = threadIdx.x % a.upr;
    const bool live = slot < nrow && unit * R < seg_len;
    float2 acc0[R], acc1[R];
#pragma unroll
    for (int r = 0; r < R; ++r) { acc0[r] = make_float2(0.f, 0.f); acc1[r] = make_float2(0.f, 0.f); }
    if (live) {
        // inputs of this thread: local indices [unit*R, unit*R + R + H), newest = unit*R + R - 1 + H
        const float2* vp = vin + (size_t)slot * in_stride + unit * R;
#pragma unroll
        for (int jj = 0; jj < R + H; ++jj) {
            const float2 v = vp[R - 1 + H - jj];                        // input i = m0 + R - 1 - jj
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int q = r - (R - 1) + jj;                         // tap pair index of position r
                if (q >= 0 && q < HALF) {
                    // packed (re, im) FMA with the tap as a broadcast uniform-register operand: half the issue
                    // slots of four scalar FFMAs, so the loads and index arithmetic issue in their shadow
                    acc0[r] = __ffma2_rn(make_float2(taps.t0[q], taps.t0[q]), v, acc0[r]);
                    acc1[r] = __ffma2_rn(make_float2(taps.t1[q], taps.t1[q]), v, acc1[r]);
                }
            }
        }
    }
    if (pre) {                                                          // every thread's cp.async has landed
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();
    }
    if (live) {
        float2* op = vout + (size_t)slot * out_stride + 2 * unit * R;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            float2 w0 = make_float2(2.f * acc0[r].x, 2.f * acc0[r].y), w1 = make_float2(2.f * acc1[r].x, 2.f * acc1[r].y);
            if (pre && unit * R + r < seg_len) {
                const float2 p0 = op[2 * r], p1 = op[2 * r + 1];
                w0.x += p0.x; w0.y += p0.y; w1.x += p1.x; w1.y += p1.y;
            }
            op[2 * r] = w0;
            op[2 * r + 1] = w1;
        }
    }
    __syncthreads();

    // coalesced write-out (16-byte accesses: even complex index, out rows are 16-byte aligned)
#pragma unroll 4
    for (int sl = 0; sl < nrow; ++sl) {
        float4* o = reinterpret_cast<float4*>(a.out + (size_t)(row0 + sl) * 2 * a.n_in + 2 * m_base);
        const float4* src = reinterpret_cast<const float4*>(vout + (size_t)sl * out_stride);
        for (int i = threadIdx.x; i < seg_len; i += blockDim.x) {
            float4 w = src[i];
            if (a.accumulate && !pre) { const float4 p = o[i]; w.x += p.x; w.y += p.y; w.z += p.z; w.w += p.w; }
            o[i] = w;
        }
    }
    // carried history: last H inputs of hist ++ in (written with the first segment of a row)
    if (seg_idx == 0 && H > 0) {
#pragma unroll 4
        for (int sl = 0; sl < nrow; ++sl) {
            const int row = row0 + sl;
            for (int i = threadIdx.x; i < H; i += blockDim.x) {
                const int g = a.n_in - H + i;
                hnext[(size_t)row * H + i] = (g >= 0) ? a.in[(size_t)row * a.n_in + g] : hcur[(size_t)row * H + a.n_in + i];
            }
        }
    }
    if (last_cta_arrives(a.phase, gridDim.x)) a.phase[0] = ph ^ 1;
}

// ---------------------------------------------------------------------------------------------
// Streaming up-by-2 (+ accumulate) for SHORT filters (32 taps: 32 FMA per 20 bytes, HBM-bound).
//
// No shared memory and no CTA-wide phases: a thread owns R = 4 consecutive input positions, reads the
// R + HALF inputs it needs as 16-byte loads straight from global memory (neighbouring threads overlap,
// the L1 serves the re-reads), fetches the 8 outputs it accumulates into, and writes 8 outputs.  With
// ~100 bytes of DRAM traffic in flight per thread and 1024+ threads per SM the memory system stays busy
// without any staging.  Taps are kernel parameters (constant bank).
// ---------------------------------------------------------------------------------------------
constexpr int kUpSR = 4;

template <int HALF>
__global__ void __launch_bounds__(256) spiir_up2_stream_kernel(const UpArgs a, const __grid_constant__ UpTaps<HALF> taps)
{
    constexpr int R = kUpSR, H = HALF - 1;
    static_assert(HALF % 2 == 0, "the aligned fast path reads HALF + R inputs as pairs");
    const int ph = phase_read(a.phase);
    const float2* hcur = a.hbuf[ph];
    float2* hnext = a.hbuf[ph ^ 1];
    const int upr = (a.n_in + R - 1) / R;                                // units per row
    const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int row = (int)(id / upr), unit = (int)(id - (long long)row * upr);
    if (row < a.rows) {
        const int m0 = unit * R;
        const float2* in = a.in + (size_t)row * a.n_in;
        float2 v[R + HALF];                                             // v[i] = input m0 - HALF + i  (v[0] unused by the FIR)
        if (m0 >= HALF && m0 + R <= a.n_in && (a.n_in & 1) == 0) {
            const float4* p = reinterpret_cast<const float4*>(in + m0 - HALF);
#pragma unroll
            for (int i = 0; i < (R + HALF) / 2; ++i) {
                const float4 q = p[i];
                v[2 * i] = make_float2(q.x, q.y);
                v[2 * i + 1] = make_float2(q.z, q.w);
            }
        } else {
            const float2* hist = hcur + (size_t)row * H;
#pragma unroll
            for (int i = 0; i < R + HALF; ++i) {
                const int g = m0 - HALF + i;
                float2 x = make_float2(0.f, 0.f);
                if (g >= 0) { if (g < a.n_in) x = in[g]; }
                else if (H + g >= 0) x = hist[H + g];
                v[i] = x;
            }
        }
        float4* o = reinterpret_cast<float4*>(a.out + (size_t)row * 2 * a.n_in) + m0;
        float4 old[R];
#pragma unroll
        for (int r = 0; r < R; ++r)
            old[r] = (a.accumulate && m0 + r < a.n_in) ? o[r] : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            float2 acc0 = make_float2(0.f, 0.f), acc1 = make_float2(0.f, 0.f);
#pragma unroll
            for (int q = 0; q < HALF; ++q) {
                const float2 x = v[HALF + r - q];                       // input m0 + r - q
                acc0 = __ffma2_rn(make_float2(taps.t0[q], taps.t0[q]), x, acc0);
                acc1 = __ffma2_rn(make_float2(taps.t1[q], taps.t1[q]), x, acc1);
            }
            if (m0 + r < a.n_in)
                o[r] = make_float4(fmaf(2.f, acc0.x, old[r].x), fmaf(2.f, acc0.y, old[r].y),
                                   fmaf(2.f, acc1.x, old[r].z), fmaf(2.f, acc1.y, old[r].w));
        }
        // carried history: the first H units of a row copy one sample each (last H inputs of hist ++ in)
        if (H > 0) {
            for (int i = unit; i < H; i += upr) {
                const int g = a.n_in - H + i;
                hnext[(size_t)row * H + i] = (g >= 0) ? in[g] : hcur[(size_t)row * H + a.n_in + i];
            }
        }
    }
    if (last_cta_arrives(a.phase, gridDim.x)) a.phase[0] = ph ^ 1;
}

// ---------------------------------------------------------------------------------------------
// Register-blocked down-by-2 for a compile-time tap count N (real rows).
//
// A thread owns R = 10 consecutive outputs; they depend on N + 2R - 2 consecutive inputs, fetched
// with 16-byte LDS (four inputs feed up to 4R FFMAs).  Lane l starts at word 2R*l = 20 l, i.e. five
// 16-byte chunks apart: 5 is odd, so the eight lanes of an LDS.128 phase hit eight different bank
// groups.  Taps are kernel parameters (constant bank -> uniform registers), loop fully unrolled.
// w[i] = u[2*m_base - (N-1) + i] is the staged input (history first); output ml of the segment is
// sum_j h[j] * w[2*ml + N-1 - j].
// ---------------------------------------------------------------------------------------------
constexpr int kDownR = 10;
constexpr int kDownSegMax = 128 * kDownR;              // outputs per row segment of the standalone kernel

template <int N>
struct DownTaps { float h[N]; };

template <int N, int R = kDownR>
__device__ __forceinline__ void down2_units(const float* __restrict__ w, int n_out, float* __restrict__ out_s,
                                            const DownTaps<N>& taps, int first_unit, int unit_stride)
{
    static_assert(R % 2 == 0, "a unit starts at word 2 R unit: 16-byte aligned only for even R");
    constexpr int NIN = N + 2 * R - 2, NLD = (NIN + 3) / 4;
    for (int unit = first_unit; unit * R < n_out; unit += unit_stride) {
        const float4* wp = reinterpret_cast<const float4*>(w + 2 * unit * R);
        float acc[R];
#pragma unroll
        for (int r = 0; r < R; ++r) acc[r] = 0.f;
#pragma unroll
        for (int c = 0; c < NLD; ++c) {
            const float4 v = wp[c];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int ii = 4 * c + e;                               // input index relative to the unit
                const float x = e == 0 ? v.x : e == 1 ? v.y : e == 2 ? v.z : v.w;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int j = 2 * r + N - 1 - ii;                   // tap of output r for this input
                    if (ii < NIN && j >= 0 && j < N) acc[r] = fmaf(taps.h[j], x, acc[r]);
                }
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (unit * R + r < n_out) out_s[unit * R + r] = acc[r];
    }
}

struct DownArgs {
    const float* in;         // [rows][n_in]
    float*       out;        // [rows][n_in/2]
    float*       hbuf[2];    // [rows][N-1] ping-pong, hbuf[phase] is current
    int*         phase;
    int rows, n_in;
    int seg;                 // outputs per row segment (multiple of 2, <= kDownSegMax)
    int nseg;
};

// R outputs per thread: 6 for 192 and 384 taps, 10 for 32.  The fully unrolled body is R x N FFMAs; at 384 taps and
// R = 10 (61 KB of code) the kernel ran at the speed of its instruction-cache misses (3.65 ms for 16384 x 4096 -> 2048
// against 0.65 ms at R = 6).  R = 4 and 8 put the lanes' 16-byte loads 2 or 4 chunks apart: bank conflicts.
template <int N, int R = kDownR>
__global__ void __launch_bounds__(128, 8) spiir_down2_fir_kernel(const DownArgs a, const __grid_constant__ DownTaps<N> taps)
{
    constexpr int H = N - 1;
    extern __shared__ __align__(16) float smd[];
    const int seg_idx = blockIdx.x % a.nseg, row = blockIdx.x / a.nseg;
    const int n_out = a.n_in >> 1;
    const int m_base = seg_idx * a.seg;
    const int seg_len = min(a.seg, n_out - m_base);
    const int w_len = (2 * a.seg + H + 2 * R + 7) & ~3;                // staged inputs incl. over-read pad
    float* w = smd;
    float* out_s = smd + w_len;
    const int ph = phase_read(a.phase);
    const float* in = a.in + (size_t)row * a.n_in;
    const float* hist = a.hbuf[ph] + (size_t)row * H;
    // eight independent loads in flight per thread (a rolled loop keeps one: 21 DRAM round trips in a row per CTA;
    // 192 taps: 472 -> 362 us)
    for (int i0 = threadIdx.x; i0 < w_len; i0 += 8 * blockDim.x) {
        float v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int i = i0 + k * blockDim.x;
            const int g = 2 * m_base - H + i;
            v[k] = 0.f;
            if (i < 2 * seg_len + H) {
                if (g >= 0) v[k] = in[g];
                else if (H + g >= 0) v[k] = hist[H + g];
            }
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int i = i0 + k * blockDim.x;
            if (i < w_len) w[i] = v[k];
        }
    }
    __syncthreads();
    down2_units<N, R>(w, seg_len, out_s, taps, threadIdx.x, blockDim.x);
    __syncthreads();
    float* o = a.out + (size_t)row * n_out + m_base;
    for (int i = threadIdx.x; i < seg_len; i += blockDim.x) o[i] = out_s[i];
    if (seg_idx == 0) {
        float* hn = a.hbuf[ph ^ 1] + (size_t)row * H;
        for (int i = threadIdx.x; i < H; i += blockDim.x) {
            const int g = a.n_in - H + i;
            hn[i] = (g >= 0) ? in[g] : hist[a.n_in + i];
        }
    }
    if (last_cta_arrives(a.phase, gridDim.x)) a.phase[0] = ph ^ 1;
}

// ---------------------------------------------------------------------------------------------
// Whole down chain of the multirate plan in one launch (row a8): one CTA per stream runs the
// stages one after the other out of shared memory.  Buffer of stage h: [history (N-1) | data n_h],
// which is exactly the w[] layout of down2_units with m_base = 0; the outputs of a stage are the
// data part of the next buffer and also go to global memory (the banks read them there).
// ---------------------------------------------------------------------------------------------
constexpr int kMaxStages = 15;
struct DownChainArgs {
    const float* x;                  // [S][n] base-rate input
    float*       xh[kMaxStages];     // xh[k]: [S][n >> (k+1)] output of stage k
    float*       hbuf[kMaxStages][2];   // [S][N-1] per stage, ping-pong
    int*         phase[kMaxStages];     // per stage {phase, arrivals}; arrivals of stage 0 count this kernel's CTAs
    int n, nstages;
};

__device__ __forceinline__ int ph_of(const int (&ph)[15], int k)
{
    int v = 0;
#pragma unroll
    for (int i = 0; i < 15; ++i) v = (i == k) ? ph[i] : v;
    return v;
}
constexpr int kChainPad = 32;        // zeroed words after a buffer (the 16-byte loads of the last unit over-read)
__host__ __device__ inline int down_chain_buf_len(int N, int n_in) { return (N - 1 + n_in + kChainPad + 3) & ~3; }

template <int N>
__global__ void __launch_bounds__(512) spiir_down_chain_kernel(const DownChainArgs a, const __grid_constant__ DownTaps<N> taps)
{
    constexpr int H = N - 1;
    extern __shared__ __align__(16) float smd[];
    const int s = blockIdx.x;
    float* w = smd;                                                     // [history H | data n_in | pad]
    int ph[kMaxStages];
    {   // Every stage's history and zero pad, and the caller's block, up front.  All phase words are read first, then all
        // history words of this thread are fetched before any of them is stored: two DRAM round trips in total instead
        // of two per stage.
#pragma unroll
        for (int k = 0; k < kMaxStages; ++k) ph[k] = k < a.nstages ? phase_read(a.phase[k]) : 0;
        const float* __restrict__ xr = a.x + (size_t)s * a.n;
        float hv[kMaxStages];
#pragma unroll
        for (int k = 0; k < kMaxStages; ++k)
            hv[k] = (k < a.nstages && (int)threadIdx.x < H) ? a.hbuf[k][ph[k]][(size_t)s * H + threadIdx.x] : 0.f;
        static_assert(H <= 512, "one history word per thread and stage");
        float* wk = smd;
        int n_k = a.n;
#pragma unroll
        for (int k = 0; k < kMaxStages; ++k) {
            if (k < a.nstages) {
                const int len = down_chain_buf_len(N, n_k);
                if ((int)threadIdx.x < H) wk[threadIdx.x] = hv[k];
                for (int i = H + n_k + threadIdx.x; i < len; i += blockDim.x) wk[i] = 0.f;
                if (k == 0) {
                    float* wd = wk + H;
#pragma unroll 8
                    for (int i = threadIdx.x; i < n_k; i += blockDim.x) wd[i] = xr[i];
                }
                wk += len; n_k >>= 1;
            }
        }
    }
    int n_in = a.n;
    for (int k = 0; k < a.nstages; ++k) {
        const int n_out = n_in >> 1;
        float* wn = w + down_chain_buf_len(N, n_in);                    // buffer of the next stage
        __syncthreads();
        // outputs per thread: as few as keep all threads busy (a thread's FIR is a serial chain of N R FMAs)
        if (n_out > 4 * (int)blockDim.x) down2_units<N, kDownR>(w, n_out, wn + H, taps, threadIdx.x, blockDim.x);
        else if (n_out > 2 * (int)blockDim.x) down2_units<N, 4>(w, n_out, wn + H, taps, threadIdx.x, blockDim.x);
        else down2_units<N, 2>(w, n_out, wn + H, taps, threadIdx.x, blockDim.x);
        __syncthreads();
        float* o = a.xh[k] + (size_t)s * n_out;
        for (int i = threadIdx.x; i < n_out; i += blockDim.x) o[i] = wn[H + i];
        // carried history of stage k: the last H words of [history | data]
        float* hn = a.hbuf[k][ph_of(ph, k) ^ 1] + (size_t)s * H;
        for (int i = threadIdx.x; i < H; i += blockDim.x) hn[i] = w[n_in + i];
        w = wn; n_in = n_out;
    }
    if (last_cta_arrives(a.phase[0], gridDim.x))
        for (int k = 0; k < a.nstages; ++k) a.phase[k][0] ^= 1;
}

// ---------------------------------------------------------------------------------------------
// Whole up-and-accumulate cascade of the multirate plan in one launch (row a10).  One CTA per
// (stream, template) row climbs from the lowest rate to the base rate:
//     acc = z_low;   for every stage: acc <- z_add[stage] + up2(acc);   out = last acc.
// The running acc never leaves shared memory (two buffers that swap roles; buffer of a stage =
// [history (HALF-1) | data n_in | zero pad]), only the per-rate SNR series are read from global and
// only the base-rate result is written.  The FIR of a stage is the register-blocked loop of
// spiir_up2_fir_kernel; the ten z_add values a thread adds to are fetched before its FIR loop, so
// their latency hides behind ~2000 FFMAs.  z_add of the last stage may alias `out` (in place).
// ---------------------------------------------------------------------------------------------
struct UpChainArgs {
    const float2* z_low;                 // [rows][n_low] output of the lowest-rate bank
    const float2* z_add[kMaxStages];     // stage k: [rows][2 * (n_low << k)]
    float2*       out;                   // [rows][n_low << nstages]
    float2*       hbuf[kMaxStages][2];   // stage k: [rows][HALF-1], ping-pong
    int*          phase[kMaxStages];     // per stage {phase, arrivals}; arrivals of stage 0 count this kernel's CTAs
    int rows, n_low, nstages;
    int cap_a, cap_b;                    // complex words of the two buffers
};

__host__ __device__ inline int up_chain_buf_len(int half, int n_in) { return (half - 1 + n_in + kUpR + 4) & ~1; }

template <int HALF>
__global__ void __launch_bounds__(128, 7) spiir_up_chain_kernel(const UpChainArgs a, const __grid_constant__ UpTaps<HALF> taps)
{
    constexpr int R = kUpR, H = HALF - 1;
    extern __shared__ __align__(16) float2 smu[];
    const int row = blockIdx.x;
    // stage k reads buffer (k & 1) and writes buffer ((k + 1) & 1); sizes are laid out so that the
    // buffer holding the largest input (the last stage's) is the one of parity (nstages - 1) & 1
    float2* buf[2];
    buf[(a.nstages - 1) & 1] = smu;
    buf[a.nstages & 1] = smu + a.cap_a;
    {
        float2* cur = buf[0];
        const float2* zl = a.z_low + (size_t)row * a.n_low;
        const float2* h0 = a.hbuf[0][phase_read(a.phase[0])] + (size_t)row * H;
        const int len = up_chain_buf_len(HALF, a.n_low);
        for (int i = threadIdx.x; i < len; i += blockDim.x)
            cur[i] = i < H ? h0[i] : (i < H + a.n_low ? zl[i - H] : make_float2(0.f, 0.f));
    }
    for (int k = 0; k < a.nstages; ++k) {
        const int n_in = a.n_low << k;
        const bool last = k == a.nstages - 1;
        float2* cur = buf[k & 1];
        float2* nxt = buf[(k + 1) & 1];
        if (!last) {                                                    // history and zero pad of the next buffer
            const float2* hk = a.hbuf[k + 1][phase_read(a.phase[k + 1])] + (size_t)row * H;
            const int len = up_chain_buf_len(HALF, 2 * n_in);
            for (int i = threadIdx.x; i < len; i += blockDim.x)
                if (i < H || i >= H + 2 * n_in) nxt[i] = i < H ? hk[i] : make_float2(0.f, 0.f);
        }
        __syncthreads();
        {   // carried history of this stage: the last H words of [history | data]
            float2* hn = a.hbuf[k][phase_read(a.phase[k]) ^ 1] + (size_t)row * H;
            for (int i = threadIdx.x; i < H; i += blockDim.x) hn[i] = cur[n_in + i];
        }
        const float2* zadd = a.z_add[k] + (size_t)row * 2 * n_in;
        float2* gout = a.out + (size_t)row * 2 * n_in;                  // used by the last stage only
        for (int unit = threadIdx.x; unit * R < n_in; unit += blockDim.x) {
            const int m0 = unit * R;
            float4 old[R];
#pragma unroll
            for (int r = 0; r < R; ++r)
                old[r] = m0 + r < n_in ? reinterpret_cast<const float4*>(zadd)[m0 + r] : make_float4(0.f, 0.f, 0.f, 0.f);
            const float2* vp = cur + m0;                                // inputs [m0, m0 + R + H), newest last
            float2 acc0[R], acc1[R];
#pragma unroll
            for (int r = 0; r < R; ++r) { acc0[r] = make_float2(0.f, 0.f); acc1[r] = make_float2(0.f, 0.f); }
#pragma unroll
            for (int jj = 0; jj < R + H; ++jj) {
                const float2 v = vp[R - 1 + H - jj];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int q = r - (R - 1) + jj;
                    if (q >= 0 && q < HALF) {
                        acc0[r] = __ffma2_rn(make_float2(taps.t0[q], taps.t0[q]), v, acc0[r]);
                        acc1[r] = __ffma2_rn(make_float2(taps.t1[q], taps.t1[q]), v, acc1[r]);
                    }
                }
            }
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if (m0 + r < n_in) {
                    const float4 w = make_float4(fmaf(2.f, acc0[r].x, old[r].x), fmaf(2.f, acc0[r].y, old[r].y),
                                                 fmaf(2.f, acc1[r].x, old[r].z), fmaf(2.f, acc1[r].y, old[r].w));
                    if (last) reinterpret_cast<float4*>(gout)[m0 + r] = w;
                    else { nxt[H + 2 * (m0 + r)] = make_float2(w.x, w.y); nxt[H + 2 * (m0 + r) + 1] = make_float2(w.z, w.w); }
                }
            }
        }
        __syncthreads();
    }
    if (last_cta_arrives(a.phase[0], gridDim.x))
        for (int k = 0; k < a.nstages; ++k) a.phase[k][0] ^= 1;
}

}  // namespace spiir
