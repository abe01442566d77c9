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

namespace spiir {

constexpr int kMaxTaps = 1024;

struct ResampArgs {
    const float* taps;      // [N] float32 taps (device)
    const void*  in;        // down: float [rows][n_in]; up: float2 [rows][n_in]
    void*        out;       // down: float [rows][n_in/2]; up: float2 [rows][2 n_in]
    const void*  hist;      // down: float [rows][N-1]; up: float2 [rows][N/2-1]
    void*        hist_next;
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
    const float* in = reinterpret_cast<const float*>(a.in) + (size_t)row * a.n_in;
    const float* hist = reinterpret_cast<const float*>(a.hist) + (size_t)row * H;
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
        float* hn = reinterpret_cast<float*>(a.hist_next) + (size_t)row * H;
        for (int i = threadIdx.x; i < H; i += blockDim.x) {
            const int g = a.n_in - H + i;
            hn[i] = (g >= 0) ? in[g] : hist[a.n_in + i];
        }
    }
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
    const float2* in = reinterpret_cast<const float2*>(a.in) + (size_t)row * a.n_in;
    const float2* hist = reinterpret_cast<const float2*>(a.hist) + (size_t)row * H;
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
        float2* hn = reinterpret_cast<float2*>(a.hist_next) + (size_t)row * H;
        for (int i = threadIdx.x; i < H; i += blockDim.x) {
            const int g = a.n_in - H + i;
            hn[i] = (g >= 0) ? in[g] : hist[a.n_in + i];
        }
    }
}

}  // namespace spiir
