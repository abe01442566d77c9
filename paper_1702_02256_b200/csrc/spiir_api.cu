// spiir_api.cu -- C ABI of libspiir.so: plans, launches, resamplers, multirate composition.
// See include/spiir.h for the contract of every entry point.
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <new>
#include <vector>

#include "spiir_filter.cuh"
#include "spiir_internal.h"
#include "spiir_resample.cuh"

namespace spiir {

spiir_status cuda_fail(cudaError_t e, const char* what)
{
    set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
    return e == cudaErrorMemoryAllocation ? SPIIR_ENOMEM : SPIIR_ECUDA;
}

spiir_status device_info(DeviceInfo* out)
{
    int dev = 0;
    SPIIR_CUDA(cudaGetDevice(&dev));
    out->device = dev;
    SPIIR_CUDA(cudaDeviceGetAttribute(&out->n_sm, cudaDevAttrMultiProcessorCount, dev));
    SPIIR_CUDA(cudaDeviceGetAttribute(&out->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    return SPIIR_OK;
}

// cudaFuncSetAttribute costs several microseconds of host time: raise a kernel's dynamic shared memory
// limit only when a launch needs more than any earlier one did (per device the limit only grows).
static cudaError_t ensure_smem(const void* func, int bytes)
{
    static std::mutex mu;
    static const void* funcs[256];
    static int devs[256], limits[256];
    static int nfuncs = 0;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);                 // the attribute is per device
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    for (int i = 0; i < nfuncs; ++i)
        if (funcs[i] == func && devs[i] == dev) {
            if (limits[i] >= bytes) return cudaSuccess;
            e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
            if (e == cudaSuccess) limits[i] = bytes;
            return e;
        }
    e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess && nfuncs < 256) { funcs[nfuncs] = func; devs[nfuncs] = dev; limits[nfuncs] = bytes; ++nfuncs; }
    return e;
}

// ---------------------------------------------------------------------------------------------
// kernel dispatch table: (F, LPT, NOZ) -> instantiation
// ---------------------------------------------------------------------------------------------
typedef void (*filter_kernel_t)(const FilterArgs);

template <int F, int LPT>
static filter_kernel_t pick_noz(bool noz)
{
    return noz ? (filter_kernel_t)spiir_filter_kernel<F, LPT, true> : (filter_kernel_t)spiir_filter_kernel<F, LPT, false>;
}

template <int LPT>
static filter_kernel_t pick_small(int F, bool noz)
{
    switch (F) {
        case 1: return pick_noz<1, LPT>(noz);
        case 2: return pick_noz<2, LPT>(noz);
        case 3: return pick_noz<3, LPT>(noz);
        case 4: return pick_noz<4, LPT>(noz);
    }
    return nullptr;
}

static filter_kernel_t pick_kernel(int F, int LPT, bool noz)
{
    switch (LPT) {
        case 1: return pick_small<1>(F, noz);
        case 2: return pick_small<2>(F, noz);
        case 4: return pick_small<4>(F, noz);
        case 8: return pick_small<8>(F, noz);
        case 16:
            switch (F) {
                case 2: return pick_noz<2, 16>(noz);
                case 3: return pick_noz<3, 16>(noz);
                case 4: return pick_noz<4, 16>(noz);
                case 5: return pick_noz<5, 16>(noz);
                case 6: return pick_noz<6, 16>(noz);
                case 7: return pick_noz<7, 16>(noz);
                case 8: return pick_noz<8, 16>(noz);
            }
            return nullptr;
        case 32:
            switch (F) {
                case 1: return pick_noz<1, 32>(noz);
                case 2: return pick_noz<2, 32>(noz);
                case 3: return pick_noz<3, 32>(noz);
                case 4: return pick_noz<4, 32>(noz);
                case 5: return pick_noz<5, 32>(noz);
                case 6: return pick_noz<6, 32>(noz);
                case 7: return pick_noz<7, 32>(noz);
                case 8: return pick_noz<8, 32>(noz);
                case 10: return pick_noz<10, 32>(noz);
                case 12: return pick_noz<12, 32>(noz);
                case 14: return pick_noz<14, 32>(noz);
                case 16: return pick_noz<16, 32>(noz);
            }
    }
    return nullptr;
}

spiir_status plan_geometry(const spiir_plan* p, int n, FilterGeometry* g)
{
    return compute_geometry(p->T, p->L, p->S, p->Dpad, n, p->opt_chunks, p->NC_cap, p->dev.n_sm, p->dev.smem_optin, g);
}

static void fill_filter_args(const spiir_plan* p, const float* x, int n, spiir_c64* z, int accumulate, const FilterGeometry& g,
                             FilterArgs* a)
{
    a->coef = p->d_coef; a->dly = p->d_dly; a->state = p->d_state; a->chunk_st = p->d_chunk;
    a->hbuf[0] = p->d_hist[0]; a->hbuf[1] = p->d_hist[1]; a->phase = p->d_phase;
    a->x = x; a->z = reinterpret_cast<float2*>(z);
    a->n = n; a->T = p->T; a->G = p->G; a->S = p->S; a->Dpad = p->Dpad;
    a->NT = g.NT; a->CS = g.CS; a->NC = g.NC; a->C = g.C;
    a->x_aligned = ((reinterpret_cast<uintptr_t>(x) & 15u) == 0 && (p->S == 1 || (n & 3) == 0)) ? 1 : 0;
    a->accumulate = accumulate;
    a->mode = 0;
}

spiir_status filter_launch(spiir_plan* p, const float* x, int n, spiir_c64* z, int accumulate, cudaStream_t st)
{
    FilterGeometry g;
    spiir_status rc = plan_geometry(p, n, &g);
    if (rc != SPIIR_OK) return rc;
    FilterArgs a;
    fill_filter_args(p, x, n, z, accumulate, g, &a);
    const dim3 grid(g.grid_x, g.grid_y), block(g.warps * 32);
    for (int pass = 0; pass < (g.NC > 1 ? 2 : 1); ++pass) {
        a.mode = g.NC > 1 ? pass + 1 : 0;
        filter_kernel_t k = pick_kernel(g.F, g.LPT, a.mode == 1);
        if (!k) { set_error("no kernel for F=%d LPT=%d", g.F, g.LPT); return SPIIR_EUNSUPPORTED; }
        SPIIR_CUDA(ensure_smem((const void*)k, g.smem_bytes));
        k<<<grid, block, g.smem_bytes, st>>>(a);
        SPIIR_CUDA(cudaGetLastError());
        if (a.mode == 1) {
            const int nf = (int)p->nfilt;
            spiir_chunk_carry_kernel<<<(nf + 255) / 256, 256, 0, st>>>(p->d_coef, p->d_state, p->d_chunk, nf, p->S, g.NC, g.C);
            SPIIR_CUDA(cudaGetLastError());
        }
    }
    return SPIIR_OK;
}

// Several unchunked banks with the same lane mapping in ONE launch (blockIdx.z = bank).  Returns
// SPIIR_EUNSUPPORTED when the banks do not qualify; the caller then launches them one by one.
typedef void (*multi_kernel_t)(const MultiFilterArgs);
static multi_kernel_t pick_multi(int F, int LPT)
{
    if (LPT != 32) return nullptr;
    switch (F) {
        case 1: return spiir_filter_multi_kernel<1, 32>;
        case 2: return spiir_filter_multi_kernel<2, 32>;
        case 3: return spiir_filter_multi_kernel<3, 32>;
        case 4: return spiir_filter_multi_kernel<4, 32>;
        case 5: return spiir_filter_multi_kernel<5, 32>;
        case 6: return spiir_filter_multi_kernel<6, 32>;
        case 7: return spiir_filter_multi_kernel<7, 32>;
        case 8: return spiir_filter_multi_kernel<8, 32>;
    }
    return nullptr;
}

spiir_status filter_launch_group(spiir_plan* const* ps, const float* const* xs, const int* ns, spiir_c64* const* zs, int count,
                                 cudaStream_t st)
{
    if (count < 2 || count > kMaxMulti) return SPIIR_EUNSUPPORTED;
    MultiFilterArgs m;
    int F = 0, LPT = 0, warps = 0, gx = 0, gy = 0, smem = 0;
    for (int k = 0; k < count; ++k) {
        FilterGeometry g;
        spiir_status rc = plan_geometry(ps[k], ns[k], &g);
        if (rc != SPIIR_OK) return rc;
        if (g.NC != 1) return SPIIR_EUNSUPPORTED;
        if (k == 0) { F = g.F; LPT = g.LPT; }
        else if (g.F != F || g.LPT != LPT) return SPIIR_EUNSUPPORTED;
        fill_filter_args(ps[k], xs[k], ns[k], zs[k], 0, g, &m.bank[k]);
        m.gx[k] = g.grid_x; m.gy[k] = g.grid_y;
        warps = std::max(warps, g.warps); gx = std::max(gx, g.grid_x); gy = std::max(gy, g.grid_y);
        smem = std::max(smem, g.smem_bytes);
    }
    multi_kernel_t k = pick_multi(F, LPT);
    if (!k) return SPIIR_EUNSUPPORTED;
    SPIIR_CUDA(ensure_smem((const void*)k, smem));
    k<<<dim3(gx, gy, count), warps * 32, smem, st>>>(m);
    SPIIR_CUDA(cudaGetLastError());
    return SPIIR_OK;
}

}  // namespace spiir

using namespace spiir;

extern "C" {

void spiir_plan_destroy(spiir_plan_t* p)
{
    if (!p) return;
    cudaFree(p->d_coef); cudaFree(p->d_dly); cudaFree(p->d_state); cudaFree(p->d_chunk);
    cudaFree(p->d_hist[0]); cudaFree(p->d_hist[1]); cudaFree(p->d_pos); cudaFree(p->d_phase);
    delete p;
}

spiir_status spiir_plan_create(spiir_plan_t** out, const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays,
                               int n_templates, int n_filters, int rate_hz, const spiir_plan_opts* opts)
{
    if (!out) { set_error("spiir_plan_create: out is NULL"); return SPIIR_EINVAL; }
    *out = nullptr;
    if (!a1 || !b0 || !delays || n_templates < 1 || n_filters < 1) {
        set_error("spiir_plan_create: NULL array or non-positive shape");
        return SPIIR_EINVAL;
    }
    spiir_plan_opts o = {1, 4096, 0, 0};
    if (opts) o = *opts;
    if (o.n_streams < 1 || o.max_block < 1 || o.time_chunks < 0) {
        set_error("spiir_plan_create: bad options");
        return SPIIR_EINVAL;
    }
    const size_t TL = (size_t)n_templates * n_filters;
    int dmax = 0;
    for (size_t i = 0; i < TL; ++i) {
        if (delays[i] < 0 || delays[i] >= (1 << 20)) { set_error("spiir_plan_create: delay out of range at %zu", i); return SPIIR_EINVAL; }
        dmax = std::max(dmax, (int)delays[i]);
    }
    int F, LPT;
    if (!choose_lane_mapping(n_filters, n_templates, &F, &LPT)) {
        set_error("spiir_plan_create: n_filters = %d not supported (1..512)", n_filters);
        return SPIIR_EUNSUPPORTED;
    }
    spiir_plan* p = new (std::nothrow) spiir_plan;
    if (!p) return SPIIR_ENOMEM;
    spiir_status rc = device_info(&p->dev);
    if (rc != SPIIR_OK) { delete p; return rc; }
    p->T = n_templates; p->L = n_filters; p->S = o.n_streams; p->rate_hz = rate_hz; p->max_block = o.max_block;
    p->Dmax = dmax; p->Dpad = std::max(4, (dmax + 3) / 4 * 4);
    p->F = F; p->LPT = LPT; p->TPG = 32 / LPT; p->G = (n_templates + p->TPG - 1) / p->TPG;
    p->nfilt = (size_t)p->G * F * 32;
    p->opt_chunks = o.time_chunks; p->flags = o.flags;
    // chunk scratch: sized for the geometry of the largest block, at most 256 MiB
    p->NC_cap = 1 << 20;
    FilterGeometry g;
    rc = plan_geometry(p, o.max_block, &g);
    if (rc != SPIIR_OK) { delete p; return rc; }
    int nc = g.NC;
    while (nc > 1 && (size_t)nc * p->S * p->nfilt * sizeof(float2) > ((size_t)256 << 20)) nc /= 2;
    p->NC_cap = std::max(1, nc);

    std::vector<float> coef;
    std::vector<int32_t> dly, pos;
    build_layout(a1, b0, delays, n_templates, n_filters, F, LPT, (o.flags & 1) == 0, &coef, &dly, &pos);
    p->conflict_degree = layout_conflict_degree(dly, p->G, F);

#define SPIIR_TRY(call)                                                                 \
    do {                                                                                \
        cudaError_t e__ = (call);                                                       \
        if (e__ != cudaSuccess) { spiir_status s__ = cuda_fail(e__, #call); spiir_plan_destroy(p); return s__; } \
    } while (0)
    SPIIR_TRY(cudaMalloc(&p->d_coef, p->nfilt * sizeof(float4)));
    SPIIR_TRY(cudaMalloc(&p->d_dly, p->nfilt * sizeof(int32_t)));
    SPIIR_TRY(cudaMalloc(&p->d_state, (size_t)p->S * p->nfilt * sizeof(float2)));
    SPIIR_TRY(cudaMalloc(&p->d_pos, TL * sizeof(int32_t)));
    SPIIR_TRY(cudaMalloc(&p->d_hist[0], (size_t)p->S * p->Dpad * sizeof(float)));
    SPIIR_TRY(cudaMalloc(&p->d_hist[1], (size_t)p->S * p->Dpad * sizeof(float)));
    SPIIR_TRY(cudaMalloc(&p->d_phase, 2 * sizeof(int)));
    SPIIR_TRY(cudaMemset(p->d_phase, 0, 2 * sizeof(int)));
    if (p->NC_cap > 1) SPIIR_TRY(cudaMalloc(&p->d_chunk, (size_t)p->NC_cap * p->S * p->nfilt * sizeof(float2)));
    SPIIR_TRY(cudaMemcpy(p->d_coef, coef.data(), p->nfilt * sizeof(float4), cudaMemcpyHostToDevice));
    SPIIR_TRY(cudaMemcpy(p->d_dly, dly.data(), p->nfilt * sizeof(int32_t), cudaMemcpyHostToDevice));
    SPIIR_TRY(cudaMemcpy(p->d_pos, pos.data(), TL * sizeof(int32_t), cudaMemcpyHostToDevice));
    SPIIR_TRY(cudaMemset(p->d_state, 0, (size_t)p->S * p->nfilt * sizeof(float2)));
    SPIIR_TRY(cudaMemset(p->d_hist[0], 0, (size_t)p->S * p->Dpad * sizeof(float)));
    SPIIR_TRY(cudaMemset(p->d_hist[1], 0, (size_t)p->S * p->Dpad * sizeof(float)));
    if (p->d_chunk) SPIIR_TRY(cudaMemset(p->d_chunk, 0, (size_t)p->NC_cap * p->S * p->nfilt * sizeof(float2)));
#undef SPIIR_TRY
    *out = p;
    return SPIIR_OK;
}

spiir_status spiir_filter(spiir_plan_t* p, const float* x, int n, spiir_c64* snr_out, void* cuda_stream)
{
    if (!p || n < 0) { set_error("spiir_filter: bad plan or n"); return SPIIR_EINVAL; }
    if (n == 0) return SPIIR_OK;
    if (!x || !snr_out) { set_error("spiir_filter: NULL buffer"); return SPIIR_EINVAL; }
    if (n > p->max_block) { set_error("spiir_filter: n = %d exceeds max_block = %d", n, p->max_block); return SPIIR_ESTATE; }
    if (reinterpret_cast<uintptr_t>(x) & 3u || reinterpret_cast<uintptr_t>(snr_out) & 7u) {
        set_error("spiir_filter: x must be 4-byte and snr_out 8-byte aligned");
        return SPIIR_EINVAL;
    }
    return filter_launch(p, x, n, snr_out, 0, static_cast<cudaStream_t>(cuda_stream));
}

spiir_status spiir_plan_reset(spiir_plan_t* p, void* cuda_stream)
{
    if (!p) { set_error("spiir_plan_reset: NULL plan"); return SPIIR_EINVAL; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    SPIIR_CUDA(cudaMemsetAsync(p->d_state, 0, (size_t)p->S * p->nfilt * sizeof(float2), st));
    SPIIR_CUDA(cudaMemsetAsync(p->d_hist[0], 0, (size_t)p->S * p->Dpad * sizeof(float), st));
    SPIIR_CUDA(cudaMemsetAsync(p->d_hist[1], 0, (size_t)p->S * p->Dpad * sizeof(float), st));
    SPIIR_CUDA(cudaMemsetAsync(p->d_phase, 0, 2 * sizeof(int), st));
    return SPIIR_OK;
}

spiir_status spiir_plan_launch_info(const spiir_plan_t* p, int n, int info[8])
{
    if (!p || !info || n < 1) { set_error("spiir_plan_launch_info: bad arguments"); return SPIIR_EINVAL; }
    FilterGeometry g;
    spiir_status rc = plan_geometry(p, n, &g);
    if (rc != SPIIR_OK) return rc;
    info[0] = g.F; info[1] = g.LPT; info[2] = g.warps; info[3] = g.grid_x * g.grid_y;
    info[4] = g.NC; info[5] = g.smem_bytes; info[6] = g.NT; info[7] = g.launches;
    return SPIIR_OK;
}

static spiir_status state_permute(spiir_plan_t* p, spiir_c64* user, int to_user, void* cuda_stream)
{
    if (!p || !user) { set_error("spiir_plan_get/set_state: NULL argument"); return SPIIR_EINVAL; }
    const int TL = p->T * p->L;
    spiir_state_permute_kernel<<<(TL + 255) / 256, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        p->d_state, reinterpret_cast<float2*>(user), p->d_pos, TL, (int)p->nfilt, p->S, to_user);
    SPIIR_CUDA(cudaGetLastError());
    return SPIIR_OK;
}
spiir_status spiir_plan_get_state(spiir_plan_t* p, spiir_c64* y_out, void* cuda_stream) { return state_permute(p, y_out, 1, cuda_stream); }
spiir_status spiir_plan_set_state(spiir_plan_t* p, const spiir_c64* y_in, void* cuda_stream)
{
    return state_permute(p, const_cast<spiir_c64*>(y_in), 0, cuda_stream);
}

// ---------------------------------------------------------------------------------------------
// Resamplers
// ---------------------------------------------------------------------------------------------
void spiir_resamp_destroy(spiir_resamp_t* r)
{
    if (!r) return;
    cudaFree(r->d_taps); cudaFree(r->d_hist[0]); cudaFree(r->d_hist[1]); cudaFree(r->d_phase);
    delete r;
}

spiir_status spiir_resamp_create(spiir_resamp_t** out, int direction, int n_taps, double kaiser_beta, double cutoff,
                                 int n_rows, int max_block)
{
    if (!out) { set_error("spiir_resamp_create: out is NULL"); return SPIIR_EINVAL; }
    *out = nullptr;
    if ((direction != SPIIR_DOWN2 && direction != SPIIR_UP2) || n_taps < 2 || n_taps > kMaxTaps || (n_taps & 1) ||
        n_rows < 1 || max_block < 1) {
        set_error("spiir_resamp_create: bad arguments");
        return SPIIR_EINVAL;
    }
    spiir_resamp* r = new (std::nothrow) spiir_resamp;
    if (!r) return SPIIR_ENOMEM;
    r->taps.resize(n_taps);
    spiir_status rc = kaiser_taps(n_taps, kaiser_beta, cutoff, r->taps.data());
    if (rc == SPIIR_OK) rc = device_info(&r->dev);
    if (rc != SPIIR_OK) { delete r; return rc; }
    r->direction = direction; r->N = n_taps; r->rows = n_rows; r->max_block = max_block;
    r->H = direction == SPIIR_DOWN2 ? n_taps - 1 : n_taps / 2 - 1;
    const size_t hbytes = (size_t)n_rows * std::max(1, r->H) * (direction == SPIIR_DOWN2 ? sizeof(float) : sizeof(float2));
    cudaError_t e = cudaMalloc(&r->d_taps, n_taps * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&r->d_hist[0], hbytes);
    if (e == cudaSuccess) e = cudaMalloc(&r->d_hist[1], hbytes);
    if (e == cudaSuccess) e = cudaMalloc(&r->d_phase, 2 * sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(r->d_phase, 0, 2 * sizeof(int));
    if (e == cudaSuccess) e = cudaMemcpy(r->d_taps, r->taps.data(), n_taps * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemset(r->d_hist[0], 0, hbytes);
    if (e == cudaSuccess) e = cudaMemset(r->d_hist[1], 0, hbytes);
    if (e != cudaSuccess) { rc = cuda_fail(e, "spiir_resamp_create allocation"); spiir_resamp_destroy(r); return rc; }
    *out = r;
    return SPIIR_OK;
}

spiir_status spiir_resamp_reset(spiir_resamp_t* r, void* cuda_stream)
{
    if (!r) { set_error("spiir_resamp_reset: NULL"); return SPIIR_EINVAL; }
    const size_t hbytes = (size_t)r->rows * std::max(1, r->H) * (r->direction == SPIIR_DOWN2 ? sizeof(float) : sizeof(float2));
    SPIIR_CUDA(cudaMemsetAsync(r->d_hist[0], 0, hbytes, static_cast<cudaStream_t>(cuda_stream)));
    SPIIR_CUDA(cudaMemsetAsync(r->d_hist[1], 0, hbytes, static_cast<cudaStream_t>(cuda_stream)));
    SPIIR_CUDA(cudaMemsetAsync(r->d_phase, 0, 2 * sizeof(int), static_cast<cudaStream_t>(cuda_stream)));
    return SPIIR_OK;
}

spiir_status spiir_resample_down(spiir_resamp_t* r, const float* in, int n_in, float* out, void* cuda_stream)
{
    if (!r || r->direction != SPIIR_DOWN2 || n_in < 0 || (n_in & 1)) { set_error("spiir_resample_down: bad plan or odd n_in"); return SPIIR_EINVAL; }
    if (n_in == 0) return SPIIR_OK;
    if (!in || !out) { set_error("spiir_resample_down: NULL buffer"); return SPIIR_EINVAL; }
    if (n_in > r->max_block) { set_error("spiir_resample_down: n_in exceeds max_block"); return SPIIR_ESTATE; }
    if (r->N == 192 || r->N == 32) {
        // register-blocked kernel, taps in the kernel parameters (constant bank)
        DownArgs d;
        d.in = in; d.out = out;
        d.hbuf[0] = reinterpret_cast<float*>(r->d_hist[0]); d.hbuf[1] = reinterpret_cast<float*>(r->d_hist[1]);
        d.phase = r->d_phase;
        d.rows = r->rows; d.n_in = n_in;
        const int n_out = n_in / 2;
        d.nseg = (n_out + kDownSegMax - 1) / kDownSegMax;
        d.seg = ((n_out + d.nseg - 1) / d.nseg + kDownR - 1) / kDownR * kDownR;
        d.nseg = (n_out + d.seg - 1) / d.seg;
        const int w_len = (2 * d.seg + r->N - 1 + 2 * kDownR + 7) & ~3;
        const size_t smem = (size_t)(w_len + d.seg) * sizeof(float);
        const dim3 grid(d.nseg * r->rows);
        cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
        if (r->N == 192) {
            DownTaps<192> t;
            memcpy(t.h, r->taps.data(), sizeof t.h);
            spiir_down2_fir_kernel<192><<<grid, 128, smem, st>>>(d, t);
        } else {
            DownTaps<32> t;
            memcpy(t.h, r->taps.data(), sizeof t.h);
            spiir_down2_fir_kernel<32><<<grid, 128, smem, st>>>(d, t);
        }
        SPIIR_CUDA(cudaGetLastError());
        return SPIIR_OK;
    }
    ResampArgs a;
    a.taps = r->d_taps; a.in = in; a.out = out; a.hbuf[0] = r->d_hist[0]; a.hbuf[1] = r->d_hist[1]; a.phase = r->d_phase;
    a.rows = r->rows; a.n_in = n_in; a.N = r->N; a.accumulate = 0;
    const int n_out = n_in / 2;
    a.tile = std::min(512, (n_out + 127) / 128 * 128);
    const dim3 grid(r->rows, (n_out + a.tile - 1) / a.tile);
    const size_t smem = (size_t)(r->N + 2 * (a.tile + r->N / 2)) * sizeof(float);
    spiir_down2_kernel<<<grid, 128, smem, static_cast<cudaStream_t>(cuda_stream)>>>(a);
    SPIIR_CUDA(cudaGetLastError());
    return SPIIR_OK;
}

spiir_status spiir_resample_up(spiir_resamp_t* r, const spiir_c64* in, int n_in, spiir_c64* out, int accumulate,
                               void* cuda_stream)
{
    if (!r || r->direction != SPIIR_UP2 || n_in < 0) { set_error("spiir_resample_up: bad plan or n_in"); return SPIIR_EINVAL; }
    if (n_in == 0) return SPIIR_OK;
    if (!in || !out) { set_error("spiir_resample_up: NULL buffer"); return SPIIR_EINVAL; }
    if (n_in > r->max_block) { set_error("spiir_resample_up: n_in exceeds max_block"); return SPIIR_ESTATE; }
    if (reinterpret_cast<uintptr_t>(out) & 15u || reinterpret_cast<uintptr_t>(in) & 7u) {
        set_error("spiir_resample_up: out must be 16-byte and in 8-byte aligned");
        return SPIIR_EINVAL;
    }
    if (r->N == 32) {
        // short filter: HBM-bound streaming kernel, no shared memory
        UpArgs u;
        u.in = reinterpret_cast<const float2*>(in); u.out = reinterpret_cast<float2*>(out);
        u.hbuf[0] = reinterpret_cast<float2*>(r->d_hist[0]); u.hbuf[1] = reinterpret_cast<float2*>(r->d_hist[1]);
        u.phase = r->d_phase;
        u.rows = r->rows; u.n_in = n_in; u.accumulate = accumulate;
        u.seg = u.nseg = u.upr = u.rpc = 0;
        const long long units = (long long)r->rows * ((n_in + kUpSR - 1) / kUpSR);
        UpTaps<16> t;
        for (int q = 0; q < 16; ++q) { t.t0[q] = r->taps[2 * q]; t.t1[q] = r->taps[2 * q + 1]; }
        spiir_up2_stream_kernel<16><<<(unsigned)((units + 255) / 256), 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(u, t);
        SPIIR_CUDA(cudaGetLastError());
        return SPIIR_OK;
    }
    if (r->N == 192 || r->N == 32) {
        // register-blocked kernel, taps in the kernel parameters (constant bank)
        UpArgs u;
        u.in = reinterpret_cast<const float2*>(in); u.out = reinterpret_cast<float2*>(out);
        u.hbuf[0] = reinterpret_cast<float2*>(r->d_hist[0]); u.hbuf[1] = reinterpret_cast<float2*>(r->d_hist[1]);
        u.phase = r->d_phase;
        u.rows = r->rows; u.n_in = n_in; u.accumulate = accumulate;
        u.nseg = (n_in + kUpSegMax - 1) / kUpSegMax;
        u.seg = ((n_in + u.nseg - 1) / u.nseg + kUpR - 1) / kUpR * kUpR;
        u.nseg = (n_in + u.seg - 1) / u.seg;
        u.upr = u.seg / kUpR;
        u.rpc = std::max(1, std::min(128 / u.upr, r->rows));
        const int half = r->N / 2;
        const int in_stride = (u.seg + half - 1 + kUpR + 3) & ~1, out_stride = 2 * (u.seg + kUpR);
        const size_t smem = (size_t)u.rpc * (in_stride + out_stride) * sizeof(float2);
        const dim3 grid(u.nseg * ((r->rows + u.rpc - 1) / u.rpc));
        cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
        if (half == 96) {
            UpTaps<96> t;
            for (int q = 0; q < 96; ++q) { t.t0[q] = r->taps[2 * q]; t.t1[q] = r->taps[2 * q + 1]; }
            spiir_up2_fir_kernel<96><<<grid, 128, smem, st>>>(u, t);
        } else {
            UpTaps<16> t;
            for (int q = 0; q < 16; ++q) { t.t0[q] = r->taps[2 * q]; t.t1[q] = r->taps[2 * q + 1]; }
            spiir_up2_fir_kernel<16><<<grid, 128, smem, st>>>(u, t);
        }
        SPIIR_CUDA(cudaGetLastError());
        return SPIIR_OK;
    }
    ResampArgs a;
    a.taps = r->d_taps; a.in = in; a.out = out; a.hbuf[0] = r->d_hist[0]; a.hbuf[1] = r->d_hist[1]; a.phase = r->d_phase;
    a.rows = r->rows; a.n_in = n_in; a.N = r->N; a.accumulate = accumulate;
    a.tile = std::min(512, (n_in + 127) / 128 * 128);
    const dim3 grid(r->rows, (n_in + a.tile - 1) / a.tile);
    const size_t smem = (size_t)r->N * sizeof(float) + (size_t)(a.tile + r->N / 2) * sizeof(float2);
    spiir_up2_kernel<<<grid, 128, smem, static_cast<cudaStream_t>(cuda_stream)>>>(a);
    SPIIR_CUDA(cudaGetLastError());
    return SPIIR_OK;
}


// ---------------------------------------------------------------------------------------------
// FP32 FMA peak probe (measurement aid for bench.py's ALU roofline; not on the hot path): every thread
// runs 16 independent FFMA chains; returns 2 flop x FFMAs / time of the best of 5 launches.
// ---------------------------------------------------------------------------------------------
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

}  // extern "C"

namespace spiir {

// Row a8 in one launch: every down stage of a multirate plan (N = 192 only; the caller falls back to
// one spiir_resample_down per stage when this returns SPIIR_EUNSUPPORTED).
spiir_status down_chain_launch(spiir_resamp* const* downs, int nstages, const float* x, int n, float* const* xh,
                               int n_streams, cudaStream_t st)
{
    if (nstages < 1 || nstages > kMaxStages || downs[0]->N != 192) return SPIIR_EUNSUPPORTED;
    size_t words = 0;
    for (int k = 0; k <= nstages; ++k) words += down_chain_buf_len(192, n >> k);
    const size_t smem = words * sizeof(float);
    if (smem > (size_t)downs[0]->dev.smem_optin) return SPIIR_EUNSUPPORTED;
    DownChainArgs a;
    a.x = x; a.n = n; a.nstages = nstages;
    for (int k = 0; k < nstages; ++k) {
        if (downs[k]->N != 192 || downs[k]->rows != n_streams) return SPIIR_EUNSUPPORTED;
        a.xh[k] = xh[k];
        a.hbuf[k][0] = reinterpret_cast<float*>(downs[k]->d_hist[0]);
        a.hbuf[k][1] = reinterpret_cast<float*>(downs[k]->d_hist[1]);
        a.phase[k] = downs[k]->d_phase;
    }
    DownTaps<192> t;
    memcpy(t.h, downs[0]->taps.data(), sizeof t.h);
    SPIIR_CUDA(ensure_smem((const void*)spiir_down_chain_kernel<192>, (int)smem));
    spiir_down_chain_kernel<192><<<n_streams, 512, smem, st>>>(a, t);
    SPIIR_CUDA(cudaGetLastError());
    return SPIIR_OK;
}


// Row a10 in one launch.  ups[k] is the stage that turns the acc at n_low << k into n_low << (k+1) samples;
// z_add[k] the per-rate SNR it is added to (the last one may be `out` itself).
spiir_status up_chain_launch(spiir_resamp* const* ups, int nstages, const spiir_c64* z_low, int n_low,
                             const spiir_c64* const* z_add, spiir_c64* out, int rows, cudaStream_t st)
{
    if (nstages < 1 || nstages > kMaxStages) return SPIIR_EUNSUPPORTED;
    const int N = ups[0]->N;
    if (N != 192 && N != 32) return SPIIR_EUNSUPPORTED;
    UpChainArgs a;
    a.z_low = reinterpret_cast<const float2*>(z_low); a.out = reinterpret_cast<float2*>(out);
    a.rows = rows; a.n_low = n_low; a.nstages = nstages;
    for (int k = 0; k < nstages; ++k) {
        if (ups[k]->N != N || ups[k]->rows != rows) return SPIIR_EUNSUPPORTED;
        a.z_add[k] = reinterpret_cast<const float2*>(z_add[k]);
        a.hbuf[k][0] = reinterpret_cast<float2*>(ups[k]->d_hist[0]);
        a.hbuf[k][1] = reinterpret_cast<float2*>(ups[k]->d_hist[1]);
        a.phase[k] = ups[k]->d_phase;
    }
    a.cap_a = up_chain_buf_len(N / 2, n_low << (nstages - 1));
    a.cap_b = up_chain_buf_len(N / 2, nstages >= 2 ? n_low << (nstages - 2) : 1);
    const size_t smem = (size_t)(a.cap_a + a.cap_b) * sizeof(float2);
    if (smem > (size_t)ups[0]->dev.smem_optin) return SPIIR_EUNSUPPORTED;
    if (N == 192) {
        UpTaps<96> t;
        for (int q = 0; q < 96; ++q) { t.t0[q] = ups[0]->taps[2 * q]; t.t1[q] = ups[0]->taps[2 * q + 1]; }
        SPIIR_CUDA(ensure_smem((const void*)spiir_up_chain_kernel<96>, (int)smem));
        spiir_up_chain_kernel<96><<<rows, 128, smem, st>>>(a, t);
    } else {
        UpTaps<16> t;
        for (int q = 0; q < 16; ++q) { t.t0[q] = ups[0]->taps[2 * q]; t.t1[q] = ups[0]->taps[2 * q + 1]; }
        SPIIR_CUDA(ensure_smem((const void*)spiir_up_chain_kernel<16>, (int)smem));
        spiir_up_chain_kernel<16><<<rows, 128, smem, st>>>(a, t);
    }
    SPIIR_CUDA(cudaGetLastError());
    return SPIIR_OK;
}


// Whether the fused chains can serve a block of n base-rate samples (same conditions as the launchers).
bool down_chain_fits(spiir_resamp* const* downs, int nstages, int n)
{
    if (nstages < 1 || nstages > kMaxStages || downs[0]->N != 192) return false;
    size_t words = 0;
    for (int k = 0; k <= nstages; ++k) words += down_chain_buf_len(192, n >> k);
    return words * sizeof(float) <= (size_t)downs[0]->dev.smem_optin;
}

bool up_chain_fits(spiir_resamp* const* ups, int nstages, int n_low)
{
    if (nstages < 1 || nstages > kMaxStages) return false;
    const int N = ups[0]->N;
    if (N != 192 && N != 32) return false;
    const size_t cap = (size_t)up_chain_buf_len(N / 2, n_low << (nstages - 1)) +
                       (size_t)up_chain_buf_len(N / 2, nstages >= 2 ? n_low << (nstages - 2) : 1);
    return cap * sizeof(float2) <= (size_t)ups[0]->dev.smem_optin;
}

}  // namespace spiir
