// spiir_probe.cu -- MEASUREMENT AIDS for bench.py (include/spiir.h, last section).  Nothing here is on the hot path.
#include <cuda_runtime.h>

#include "spiir_internal.h"

namespace spiir {

// every thread runs 16 independent FFMA chains whose two other operands are shared constants
__global__ void __launch_bounds__(1024) spiir_fp32_probe_kernel(float* out, int iters, float c0, float c1)
{
    float a[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = threadIdx.x * 1e-3f + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < 16; ++i) a[i] = fmaf(a[i], c0, c1);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// Packed FFMA2 with a chosen number of distinct 32-bit register words read per instruction:
//   WORDS 3: acc = acc * s.F32 + acc      4: acc = acc * c + acc      5: acc = acc * s.F32 + d      6: acc = acc * c + d
// (acc, c, d register pairs, s a scalar; twelve independent chains with their own c, d, s so that no operand can come
// from the reuse cache).  The Eq. 7 update issues two 5-word FFMA2s per filter-sample.
constexpr int kProbeChains = 12;
template <int WORDS>
__global__ void __launch_bounds__(512) spiir_ffma2_probe_kernel(const float2* in, float2* out, long long* cyc, int iters)
{
    float2 acc[kProbeChains], c[kProbeChains], d[kProbeChains];
    float s[kProbeChains];
#pragma unroll
    for (int i = 0; i < kProbeChains; ++i) {
        acc[i] = in[threadIdx.x + i * 32]; c[i] = in[threadIdx.x + 512 + i * 32]; d[i] = in[threadIdx.x + 1024 + i * 32];
        s[i] = c[i].y;
    }
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < kProbeChains; ++i) {
                if (WORDS == 3) acc[i] = __ffma2_rn(acc[i], make_float2(s[i], s[i]), acc[i]);
                if (WORDS == 4) acc[i] = __ffma2_rn(acc[i], c[i], acc[i]);
                if (WORDS == 5) acc[i] = __ffma2_rn(acc[i], make_float2(s[i], s[i]), d[i]);
                if (WORDS == 6) acc[i] = __ffma2_rn(acc[i], c[i], d[i]);
            }
    }
    const long long t1 = clock64();
    float2 r = make_float2(0.f, 0.f);
#pragma unroll
    for (int i = 0; i < kProbeChains; ++i) { r.x += acc[i].x; r.y += acc[i].y; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

template <int WORDS>
static spiir_status run_ffma2_probe(const float2* in, float2* out, long long* cyc, int n_sm, double* cycles)
{
    const int iters = 2000, W = 4;
    long long h[1024];
    for (int r = 0; r < 2; ++r) {
        spiir_ffma2_probe_kernel<WORDS><<<n_sm, W * 128>>>(in, out, cyc, iters);
        SPIIR_CUDA(cudaDeviceSynchronize());
    }
    SPIIR_CUDA(cudaMemcpy(h, cyc, (size_t)n_sm * sizeof(long long), cudaMemcpyDeviceToHost));
    double s = 0;
    for (int i = 0; i < n_sm; ++i) s += (double)h[i];
    *cycles = s / n_sm / ((double)iters * 4 * kProbeChains * W);
    return SPIIR_OK;
}

}  // namespace spiir

using namespace spiir;

extern "C" {

spiir_status spiir_probe_fp32_peak(double* tflops_out)
{
    if (!tflops_out) { set_error("spiir_probe_fp32_peak: NULL"); return SPIIR_EINVAL; }
    DeviceInfo dev;
    spiir_status rc = device_info(&dev);
    if (rc != SPIIR_OK) return rc;
    const int blocks = dev.n_sm * 2, threads = 1024, iters = 4096;
    float* d = nullptr;
    SPIIR_CUDA(cudaMalloc(&d, (size_t)blocks * threads * sizeof(float)));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int r = 0; r < 6; ++r) {
        cudaEventRecord(e0);
        spiir_fp32_probe_kernel<<<blocks, threads>>>(d, iters, 0.999f, 1e-3f);
        cudaEventRecord(e1);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaFree(d); return cuda_fail(e, "spiir_probe_fp32_peak"); }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    const double fma = (double)blocks * threads * (double)iters * 64.0;
    *tflops_out = 2.0 * fma / (best * 1e-3) / 1e12;
    return SPIIR_OK;
}

spiir_status spiir_probe_ffma2_operands(double cycles_out[4])
{
    if (!cycles_out) { set_error("spiir_probe_ffma2_operands: NULL"); return SPIIR_EINVAL; }
    DeviceInfo dev;
    spiir_status rc = device_info(&dev);
    if (rc != SPIIR_OK) return rc;
    if (dev.n_sm > 1024) dev.n_sm = 1024;
    float2 *in = nullptr, *out = nullptr;
    long long* cyc = nullptr;
    SPIIR_CUDA(cudaMalloc(&in, 4096 * sizeof(float2)));
    SPIIR_CUDA(cudaMalloc(&out, (size_t)dev.n_sm * 512 * sizeof(float2)));
    SPIIR_CUDA(cudaMalloc(&cyc, (size_t)dev.n_sm * sizeof(long long)));
    static float2 h[4096];
    for (int i = 0; i < 4096; ++i) h[i] = make_float2(0.5f + 1e-4f * i, 0.9f - 1e-4f * i);
    cudaError_t e = cudaMemcpy(in, h, sizeof h, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        rc = run_ffma2_probe<3>(in, out, cyc, dev.n_sm, &cycles_out[0]);
        if (rc == SPIIR_OK) rc = run_ffma2_probe<4>(in, out, cyc, dev.n_sm, &cycles_out[1]);
        if (rc == SPIIR_OK) rc = run_ffma2_probe<5>(in, out, cyc, dev.n_sm, &cycles_out[2]);
        if (rc == SPIIR_OK) rc = run_ffma2_probe<6>(in, out, cyc, dev.n_sm, &cycles_out[3]);
    } else rc = cuda_fail(e, "spiir_probe_ffma2_operands");
    cudaFree(in); cudaFree(out); cudaFree(cyc);
    return rc;
}

}  // extern "C"
