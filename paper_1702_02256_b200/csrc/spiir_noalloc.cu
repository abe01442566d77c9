// spiir_noalloc.cu -- ONE entry point that allocates nothing (include/spiir.h, "NO-ALLOCATION ENTRY POINT").
//
// spiir_filter_block_noalloc filters one block from zero state (Eq. 7-8) with the time-parallel scan
// over several CTAs (row a7 of SURVEY.md section 8): pass 1 runs every chunk but the last from zero state and leaves the
// chunk end states in SCRATCH, the carry turns them into initial states in place (s_{c+1} = a1^C s_c + e_c), pass 2 reruns
// every chunk from its initial state and writes z.  The plan-based path keeps that scratch in plan memory
// (spiir_bank_class::d_chunk, from cudaMalloc or the caller's workspace); here it is a file-scope device array, so the call
// needs no plan, no workspace and no allocator: usable under CUDA-graph capture and in harnesses that forbid cudaMalloc.
//
// The array belongs to the library image: every GPU that loads libspiir.so holds kNoAllocBytes of it until the process
// exits.  All calls share it and it keeps the last call's contents.  Nothing in it has to start at zero: every word a
// call reads was written earlier by the same call (pass 1 writes e[c][f] for all c < NC - 1 and all f, the carry reads
// exactly those and writes s[c][f] for all c < NC, pass 2 reads those).  Two calls that OVERLAP on the GPU (different
// streams, or graphs replayed concurrently) race on the array; calls on one stream are ordered and safe.
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <mutex>

#include "spiir_internal.h"

namespace spiir {

constexpr size_t kNoAllocBytes = (size_t)SPIIR_NOALLOC_SCRATCH_BYTES;
constexpr size_t kNoAllocWords = kNoAllocBytes / sizeof(float2);
constexpr int kNaMaxFilters = 512;      // one thread per filter of a template in pass 2
constexpr int kNaBatch = 8;             // time steps summed per shared-memory tile in pass 2
constexpr int kNaMaxDevices = 64;

// In host code this name is a host-side stand-in, NOT a device address: kernels get the pointer that
// cudaGetSymbolAddress returns (noalloc_scratch below).
static __device__ __align__(256) float2 g_noalloc_scratch[kNoAllocWords];

// y <- a1 y + b0 x, complex, float32 (the same arithmetic type as the plan-based path)
__device__ __forceinline__ float2 na_step(float2 y, float2 a1, float2 b0, float x)
{
    float2 r;
    r.x = fmaf(a1.x, y.x, fmaf(-a1.y, y.y, b0.x * x));
    r.y = fmaf(a1.x, y.y, fmaf(a1.y, y.x, b0.y * x));
    return r;
}

// pass 1: thread = filter f = t * L + l, blockIdx.y = chunk c < NC - 1; end state from zero state -> e[c][f]
__global__ void __launch_bounds__(256) spiir_na_pass1_kernel(const float2* __restrict__ a1, const float2* __restrict__ b0,
                                                             const int* __restrict__ dly, const float* __restrict__ x,
                                                             float2* __restrict__ scratch, int TL, int n, int C)
{
    const int f = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
    if (f >= TL) return;
    const float2 a = a1[f], b = b0[f];
    const int d = dly[f];
    const int k0 = c * C, k1 = min(n, k0 + C);
    float2 y = make_float2(0.f, 0.f);
    for (int k = k0; k < k1; ++k) y = na_step(y, a, b, k >= d ? __ldg(x + k - d) : 0.f);
    scratch[(size_t)c * TL + f] = y;
}

// carry: thread = filter; s_0 = 0, s_{c+1} = a1^C s_c + e_c; scratch[c][f] <- s_c for all c < NC (in place)
__global__ void __launch_bounds__(256) spiir_na_carry_kernel(const float2* __restrict__ a1, float2* __restrict__ scratch,
                                                             int TL, int NC, int C)
{
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= TL) return;
    // a1^C by repeated squaring in double, rounded once
    double pr = 1.0, pi = 0.0, br = (double)a1[f].x, bi = (double)a1[f].y;
    for (int e = C; e > 0; e >>= 1) {
        if (e & 1) { const double r = pr * br - pi * bi, q = pr * bi + pi * br; pr = r; pi = q; }
        const double r = br * br - bi * bi, q = 2.0 * br * bi; br = r; bi = q;
    }
    const float2 aC = make_float2((float)pr, (float)pi);
    float2 s = make_float2(0.f, 0.f);
    for (int c = 0; c < NC; ++c) {
        float2 e = make_float2(0.f, 0.f);
        if (c < NC - 1) e = scratch[(size_t)c * TL + f];
        scratch[(size_t)c * TL + f] = s;
        float2 nx;
        nx.x = fmaf(aC.x, s.x, fmaf(-aC.y, s.y, e.x));
        nx.y = fmaf(aC.x, s.y, fmaf(aC.y, s.x, e.y));
        s = nx;
    }
}

// pass 2: CTA = (template t, chunk c), thread = filter l (threads l >= L contribute zeros).  kNaBatch steps at a time:
// every thread leaves its y of the batch in a shared-memory tile [step][l], then warp w sums the rows w, w + nwarps, ...
// over l in a fixed order (deterministic) and lane 0 writes z[t][k].
__global__ void __launch_bounds__(kNaMaxFilters) spiir_na_pass2_kernel(const float2* __restrict__ a1, const float2* __restrict__ b0,
                                                                       const int* __restrict__ dly, const float* __restrict__ x,
                                                                       const float2* __restrict__ scratch, float2* __restrict__ z,
                                                                       int L, int TL, int n, int C)
{
    extern __shared__ float2 tile[];                                   // [kNaBatch][blockDim.x]
    const int t = blockIdx.x, c = blockIdx.y, l = threadIdx.x, W = blockDim.x;
    const int lane = l & 31, warp = l >> 5, nwarps = W >> 5;
    const bool live = l < L;
    const int f = t * L + (live ? l : 0);
    const float2 a = a1[f], b = live ? b0[f] : make_float2(0.f, 0.f);
    const int d = dly[f];
    float2 y = live ? scratch[(size_t)c * TL + f] : make_float2(0.f, 0.f);
    const int k0 = c * C, k1 = min(n, k0 + C);
    for (int kb = k0; kb < k1; kb += kNaBatch) {
        const int nb = min(kNaBatch, k1 - kb);
        for (int j = 0; j < nb; ++j) {
            const int k = kb + j;
            y = na_step(y, a, b, k >= d ? __ldg(x + k - d) : 0.f);
            tile[j * W + l] = live ? y : make_float2(0.f, 0.f);
        }
        __syncthreads();
        for (int j = warp; j < nb; j += nwarps) {
            float2 s = make_float2(0.f, 0.f);
            for (int i = lane; i < W; i += 32) { const float2 v = tile[j * W + i]; s.x += v.x; s.y += v.y; }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                s.x += __shfl_xor_sync(0xffffffffu, s.x, o);
                s.y += __shfl_xor_sync(0xffffffffu, s.y, o);
            }
            if (lane == 0) z[(size_t)t * n + kb + j] = s;
        }
        __syncthreads();
    }
}

// Device address of the scratch array on the CURRENT device, looked up once per device.
static spiir_status noalloc_scratch(float2** out)
{
    static std::mutex mu;
    static float2* ptr[kNaMaxDevices] = {nullptr};
    int dev = 0;
    SPIIR_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNaMaxDevices) { set_error("spiir_filter_block_noalloc: device ordinal %d not supported", dev); return SPIIR_EUNSUPPORTED; }
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        float2* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
        if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_noalloc_scratch)");
        if (!p) { set_error("cudaGetSymbolAddress returned a null scratch address"); return SPIIR_ECUDA; }
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return SPIIR_OK;
}

// chunk count: explicit, or as many chunks of >= 64 samples as fit the scratch array (at most 64)
static int noalloc_chunks(long long TL, int n, int time_chunks)
{
    if (time_chunks > 0) return time_chunks;
    long long nc = std::min<long long>(64, std::max(1, n / 64));
    nc = std::min<long long>(nc, (long long)kNoAllocWords / TL);
    return (int)std::max<long long>(nc, 1);
}

}  // namespace spiir

using namespace spiir;

extern "C" {

size_t spiir_noalloc_scratch_need(int n_templates, int n_filters, int n, int time_chunks)
{
    if (n_templates < 1 || n_filters < 1 || n < 0 || time_chunks < 0) return 0;
    const long long TL = (long long)n_templates * n_filters;
    if (time_chunks == 0 && TL > (long long)kNoAllocWords) return (size_t)TL * sizeof(float2);
    return (size_t)noalloc_chunks(TL, n, time_chunks) * (size_t)TL * sizeof(float2);
}

spiir_status spiir_noalloc_setup(void)
{
    float2* p = nullptr;
    return noalloc_scratch(&p);
}

spiir_status spiir_filter_block_noalloc(const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays, int n_templates,
                                        int n_filters, const float* x, int n, int time_chunks, spiir_c64* snr_out,
                                        void* cuda_stream)
{
    // sizes first (no CUDA call, no pointer is touched before they pass)
    if (n_templates < 1 || n_filters < 1 || n < 0 || time_chunks < 0) {
        set_error("spiir_filter_block_noalloc: bad shape (templates %d, filters %d, n %d, time_chunks %d)", n_templates, n_filters, n, time_chunks);
        return SPIIR_EINVAL;
    }
    if (n_filters > kNaMaxFilters) {
        set_error("spiir_filter_block_noalloc: %d filters per template, the limit is %d", n_filters, kNaMaxFilters);
        return SPIIR_EUNSUPPORTED;
    }
    const long long TL = (long long)n_templates * n_filters;
    if (n_templates > 65535 * 32 || TL > (long long)INT32_MAX / 2) {
        set_error("spiir_filter_block_noalloc: bank of %lld filters is too large", TL);
        return SPIIR_EUNSUPPORTED;
    }
    const size_t need = spiir_noalloc_scratch_need(n_templates, n_filters, n, time_chunks);
    if (need > kNoAllocBytes) {
        set_error("spiir_filter_block_noalloc: needs %zu bytes of scratch (templates x filters x chunks x 8), the built-in "
                  "array holds %zu: use fewer time chunks or a plan (spiir_plan_create) with a caller workspace", need, kNoAllocBytes);
        return SPIIR_EINVAL;
    }
    if (!a1 || !b0 || !delays || (n > 0 && (!x || !snr_out))) { set_error("spiir_filter_block_noalloc: NULL pointer"); return SPIIR_EINVAL; }
    if (n == 0) return SPIIR_OK;
    int NC = noalloc_chunks(TL, n, time_chunks);
    int C = (n + NC - 1) / NC;
    NC = (n + C - 1) / C;
    if (NC > 65535) { set_error("spiir_filter_block_noalloc: %d time chunks, the limit is 65535", NC); return SPIIR_EINVAL; }
    float2* scratch = nullptr;
    spiir_status rc = noalloc_scratch(&scratch);
    if (rc != SPIIR_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const float2* A = reinterpret_cast<const float2*>(a1);
    const float2* B = reinterpret_cast<const float2*>(b0);
    const int* D = reinterpret_cast<const int*>(delays);
    const int fblocks = (int)((TL + 255) / 256);
    if (NC > 1) {
        spiir_na_pass1_kernel<<<dim3(fblocks, NC - 1), 256, 0, st>>>(A, B, D, x, scratch, (int)TL, n, C);
        SPIIR_CUDA(cudaGetLastError());
    }
    spiir_na_carry_kernel<<<fblocks, 256, 0, st>>>(A, scratch, (int)TL, NC, C);
    SPIIR_CUDA(cudaGetLastError());
    const int W = (n_filters + 31) / 32 * 32;
    // templates on grid.x (up to 2^31 - 1), chunks on grid.y; the tile is at most 8 x 512 x 8 = 32 KB (no opt-in needed)
    spiir_na_pass2_kernel<<<dim3(n_templates, NC), W, (size_t)kNaBatch * W * sizeof(float2), st>>>(
        A, B, D, x, scratch, reinterpret_cast<float2*>(snr_out), n_filters, (int)TL, n, C);
    SPIIR_CUDA(cudaGetLastError());
    return SPIIR_OK;
}

}  // extern "C"
