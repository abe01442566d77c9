// spiir_paper_design.cu -- COMPARISON KERNELS, not the product path (include/spiir.h, "COMPARISON KERNELS").
//
// The paper's own single-rate design restated in plain CUDA so that the new mapping can be timed
// against it on the same B200: one thread per filter; coefficients by coalesced global loads; y in a
// register across the time loop (Fig. 3); x[k - d] through the read-only data cache, __ldg (PAPER.md:116,
// 124); per-sample inner-warp sum by warp shuffle; warp partials combined by atomicAdd into the global SNR,
// the "DA" method the paper found fastest; block-based kernel for > 32 filters (one template per block of
// ceil(L/32)*32 threads), warp-based kernel for <= 32 filters (next_pow2(L) threads per template, several templates per
// warp, 256 threads per block).  It shares no code with the product kernels.
#include <cuda_runtime.h>

#include <algorithm>
#include <new>
#include <vector>

#include "spiir_internal.h"

struct spiir_pd_plan {
    int T = 0, L = 0, M = 0;          // M = threads per template
    int Dmax = 0, max_block = 0;
    float4* d_coef = nullptr;         // [T][M] (a1.re, a1.im, b0.re, b0.im), zero padded
    int32_t* d_dly = nullptr;         // [T][M]
    float2* d_y = nullptr;            // [T][M]
    float* d_hist = nullptr;          // [Dmax] the last Dmax samples, oldest first
    float* d_xbuf = nullptr;          // [Dmax + max_block] history ++ block
};

namespace spiir {

__global__ void pd_stage_kernel(float* xbuf, const float* __restrict__ hist, const float* __restrict__ x, int D, int n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < D + n) xbuf[i] = i < D ? hist[i] : x[i - D];
}

__global__ void pd_carry_kernel(float* hist, const float* __restrict__ xbuf, int D, int n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < D) hist[i] = xbuf[n + i];
}

// block-based kernel: one template per block, one filter per thread, warp partials by atomicAdd (DA)
__global__ void pd_block_kernel(const float4* __restrict__ coef, const int* __restrict__ dly, float2* ystate,
                                const float* __restrict__ xbuf, float* snr /* [T][n][2], zeroed */, int M, int D, int n)
{
    const int t = blockIdx.x, l = threadIdx.x;
    const size_t i = (size_t)t * M + l;
    const float4 c = coef[i];
    const int d = dly[i];
    float2 y = ystate[i];
    const float* xp = xbuf + D - d;
    float* out = snr + (size_t)t * n * 2;
    for (int k = 0; k < n; ++k) {
        const float x = __ldg(xp + k);
        const float yr = c.x * y.x - c.y * y.y + c.z * x;
        const float yi = c.x * y.y + c.y * y.x + c.w * x;
        y.x = yr; y.y = yi;
        float sr = yr, si = yi;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            sr += __shfl_down_sync(0xffffffffu, sr, o);
            si += __shfl_down_sync(0xffffffffu, si, o);
        }
        if ((l & 31) == 0) { atomicAdd(out + 2 * k, sr); atomicAdd(out + 2 * k + 1, si); }
    }
    ystate[i] = y;
}

// warp-based kernel: M = next_pow2(L) <= 32 threads per template, 256 threads per block, segmented shuffle sum
__global__ void pd_warp_kernel(const float4* __restrict__ coef, const int* __restrict__ dly, float2* ystate,
                               const float* __restrict__ xbuf, float2* snr /* [T][n] */, int T, int M, int D, int n)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int t = (int)(i / M), l = (int)(i % M);
    const bool live = t < T;
    const float4 c = live ? coef[i] : make_float4(0.f, 0.f, 0.f, 0.f);
    const int d = live ? dly[i] : 0;
    float2 y = live ? ystate[i] : make_float2(0.f, 0.f);
    const float* xp = xbuf + D - d;
    for (int k = 0; k < n; ++k) {
        const float x = __ldg(xp + k);
        const float yr = c.x * y.x - c.y * y.y + c.z * x;
        const float yi = c.x * y.y + c.y * y.x + c.w * x;
        y.x = yr; y.y = yi;
        float sr = yr, si = yi;
        for (int o = M >> 1; o > 0; o >>= 1) {
            sr += __shfl_down_sync(0xffffffffu, sr, o, M);
            si += __shfl_down_sync(0xffffffffu, si, o, M);
        }
        if (live && l == 0) snr[(size_t)t * n + k] = make_float2(sr, si);
    }
    if (live) ystate[i] = y;
}

}  // namespace spiir

using namespace spiir;

extern "C" {

void spiir_pd_plan_destroy(spiir_pd_plan_t* p)
{
    if (!p) return;
    cudaFree(p->d_coef); cudaFree(p->d_dly); cudaFree(p->d_y); cudaFree(p->d_hist); cudaFree(p->d_xbuf);
    delete p;
}

spiir_status spiir_pd_plan_create(spiir_pd_plan_t** out, const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays,
                                  int n_templates, int n_filters, int max_block)
{
    if (!out) { set_error("spiir_pd_plan_create: out is NULL"); return SPIIR_EINVAL; }
    *out = nullptr;
    if (!a1 || !b0 || !delays || n_templates < 1 || n_filters < 1 || n_filters > 1024 || max_block < 1) {
        set_error("spiir_pd_plan_create: bad arguments (1..1024 filters per template)");
        return SPIIR_EINVAL;
    }
    spiir_pd_plan* p = new (std::nothrow) spiir_pd_plan;
    if (!p) return SPIIR_ENOMEM;
    p->T = n_templates; p->L = n_filters; p->max_block = max_block;
    if (n_filters > 32) p->M = (n_filters + 31) / 32 * 32;
    else { p->M = 1; while (p->M < n_filters) p->M *= 2; }
    const size_t TM = (size_t)p->T * p->M;
    std::vector<float> coef(TM * 4, 0.f);
    std::vector<int32_t> dly(TM, 0);
    int dmax = 0;
    for (int t = 0; t < p->T; ++t)
        for (int l = 0; l < p->L; ++l) {
            const size_t s = (size_t)t * p->L + l, q = (size_t)t * p->M + l;
            if (delays[s] < 0 || delays[s] >= (1 << 20)) { delete p; set_error("spiir_pd_plan_create: delay out of range"); return SPIIR_EINVAL; }
            coef[q * 4 + 0] = a1[s].re; coef[q * 4 + 1] = a1[s].im; coef[q * 4 + 2] = b0[s].re; coef[q * 4 + 3] = b0[s].im;
            dly[q] = delays[s];
            dmax = std::max(dmax, (int)delays[s]);
        }
    p->Dmax = dmax;
    cudaError_t e = cudaMalloc(&p->d_coef, TM * sizeof(float4));
    if (e == cudaSuccess) e = cudaMalloc(&p->d_dly, TM * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMalloc(&p->d_y, TM * sizeof(float2));
    if (e == cudaSuccess) e = cudaMalloc(&p->d_hist, (size_t)std::max(1, dmax) * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&p->d_xbuf, ((size_t)dmax + max_block) * sizeof(float));
    if (e == cudaSuccess) e = cudaMemcpy(p->d_coef, coef.data(), TM * sizeof(float4), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(p->d_dly, dly.data(), TM * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemset(p->d_y, 0, TM * sizeof(float2));
    if (e == cudaSuccess) e = cudaMemset(p->d_hist, 0, (size_t)std::max(1, dmax) * sizeof(float));
    if (e != cudaSuccess) { spiir_status rc = cuda_fail(e, "spiir_pd_plan_create"); spiir_pd_plan_destroy(p); return rc; }
    *out = p;
    return SPIIR_OK;
}

spiir_status spiir_pd_plan_reset(spiir_pd_plan_t* p, void* cuda_stream)
{
    if (!p) { set_error("spiir_pd_plan_reset: NULL plan"); return SPIIR_EINVAL; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    SPIIR_CUDA(cudaMemsetAsync(p->d_y, 0, (size_t)p->T * p->M * sizeof(float2), st));
    SPIIR_CUDA(cudaMemsetAsync(p->d_hist, 0, (size_t)std::max(1, p->Dmax) * sizeof(float), st));
    return SPIIR_OK;
}

spiir_status spiir_pd_filter(spiir_pd_plan_t* p, const float* x, int n, spiir_c64* snr_out, void* cuda_stream)
{
    if (!p || n < 0) { set_error("spiir_pd_filter: bad plan or n"); return SPIIR_EINVAL; }
    if (n == 0) return SPIIR_OK;
    if (!x || !snr_out) { set_error("spiir_pd_filter: NULL buffer"); return SPIIR_EINVAL; }
    if (n > p->max_block) { set_error("spiir_pd_filter: n exceeds max_block"); return SPIIR_ESTATE; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int D = p->Dmax;
    pd_stage_kernel<<<(D + n + 255) / 256, 256, 0, st>>>(p->d_xbuf, p->d_hist, x, D, n);
    SPIIR_CUDA(cudaGetLastError());
    if (p->L > 32) {
        SPIIR_CUDA(cudaMemsetAsync(snr_out, 0, (size_t)p->T * n * sizeof(spiir_c64), st));
        pd_block_kernel<<<p->T, p->M, 0, st>>>(p->d_coef, p->d_dly, p->d_y, p->d_xbuf, reinterpret_cast<float*>(snr_out), p->M, D, n);
    } else {
        const size_t threads = (size_t)p->T * p->M;
        pd_warp_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(p->d_coef, p->d_dly, p->d_y, p->d_xbuf,
                                                                         reinterpret_cast<float2*>(snr_out), p->T, p->M, D, n);
    }
    SPIIR_CUDA(cudaGetLastError());
    if (D > 0) {
        pd_carry_kernel<<<(D + 255) / 256, 256, 0, st>>>(p->d_hist, p->d_xbuf, D, n);
        SPIIR_CUDA(cudaGetLastError());
    }
    return SPIIR_OK;
}

}  // extern "C"
