// spiir_api.cu -- C ABI of libspiir.so, part 1: single-rate banks (uniform and ragged), their device
// workspace, launches and resume state.  See include/spiir.h for the contract of every entry point.
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <mutex>
#include <new>
#include <vector>

#include "spiir_filter.cuh"
#include "spiir_internal.h"

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
// limit only when a launch needs more than any earlier one did (per device the limit only grows); the first call for a
// kernel also fixes its shared-memory carveout.
cudaError_t ensure_smem(const void* func, int bytes)
{
    static std::mutex mu;
    static const void* funcs[512];
    static int devs[512], limits[512];
    static int nfuncs = 0;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);                 // the attributes are per device
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    int slot = -1;
    for (int i = 0; i < nfuncs; ++i)
        if (funcs[i] == func && devs[i] == dev) { slot = i; break; }
    if (slot < 0) {
        // First launch of this kernel on this device: every kernel of the library asks for the SAME shared-memory carveout
        // (the maximum).  Kernels whose preferred L1 / shared split differs do not share an SM, and the multirate plan runs
        // its per-rate banks side by side on forked streams: with the default (per-kernel) carveouts they ran one after the
        // other (109 us for the six lower banks of configs[3] = the sum of their times).
        e = cudaFuncSetAttribute(func, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
        if (e != cudaSuccess) return e;
        if (nfuncs >= 512) return bytes <= 48 * 1024 ? cudaSuccess : cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
        slot = nfuncs++;
        funcs[slot] = func; devs[slot] = dev; limits[slot] = 48 * 1024;
    }
    if (bytes <= limits[slot]) return cudaSuccess;
    e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) limits[slot] = bytes;
    return e;
}

spiir_status arena_open(Arena* a, void* workspace, size_t workspace_bytes, size_t need, const char* who)
{
    a->used = 0;
    if (workspace) {
        if (reinterpret_cast<uintptr_t>(workspace) & 255u) { set_error("%s: workspace must be 256-byte aligned", who); return SPIIR_EINVAL; }
        if (workspace_bytes < need) {
            set_error("%s: workspace of %zu bytes is too small (%zu needed)", who, workspace_bytes, need);
            return SPIIR_ENOMEM;
        }
        a->base = static_cast<char*>(workspace); a->cap = workspace_bytes; a->owned = false;
        return SPIIR_OK;
    }
    void* q = nullptr;
    SPIIR_CUDA(cudaMalloc(&q, std::max<size_t>(need, 256)));
    a->base = static_cast<char*>(q); a->cap = need; a->owned = true;
    return SPIIR_OK;
}

void arena_close(Arena* a)
{
    if (a->owned && a->base) cudaFree(a->base);
    a->base = nullptr; a->owned = false;
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

template <int F>
static filter_kernel_t pick_multi_warp(bool noz)
{
    return noz ? (filter_kernel_t)spiir_filter_kernel<F, 32, true, true> : (filter_kernel_t)spiir_filter_kernel<F, 32, false, true>;
}

static filter_kernel_t pick_kernel(int F, int LPT, int NP, bool noz)
{
    if (NP > 1) {                                         // templates of more than 512 filters: NP warps x F <= 8
        if (LPT != 32) return nullptr;
        switch (F) {
            case 5: return pick_multi_warp<5>(noz);
            case 6: return pick_multi_warp<6>(noz);
            case 7: return pick_multi_warp<7>(noz);
            case 8: return pick_multi_warp<8>(noz);
        }
        return nullptr;
    }
    switch (LPT) {
        case 1: return pick_small<1>(F, noz);
        case 2: return pick_small<2>(F, noz);
        case 4: return pick_small<4>(F, noz);
        case 8:
            switch (F) {
                case 5: return pick_noz<5, 8>(noz);
                case 6: return pick_noz<6, 8>(noz);
                case 7: return pick_noz<7, 8>(noz);
                case 8: return pick_noz<8, 8>(noz);
            }
            return pick_small<8>(F, noz);
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

template <int LPT>
static filter_kernel_t pick_scan_f(int F)
{
    switch (F) {
        case 1: return (filter_kernel_t)spiir_filter_scan_kernel<1, LPT>;
        case 2: return (filter_kernel_t)spiir_filter_scan_kernel<2, LPT>;
        case 3: return (filter_kernel_t)spiir_filter_scan_kernel<3, LPT>;
        case 4: return (filter_kernel_t)spiir_filter_scan_kernel<4, LPT>;
    }
    return nullptr;
}

static filter_kernel_t pick_scan_kernel(int F, int LPT)
{
    switch (LPT) {
        case 1: return pick_scan_f<1>(F);
        case 2: return pick_scan_f<2>(F);
        case 4: return pick_scan_f<4>(F);
        case 8: return pick_scan_f<8>(F);
    }
    return nullptr;
}

spiir_status plan_geometry(const spiir_plan* p, const spiir_bank_class& c, int n, FilterGeometry* g)
{
    return compute_geometry(c.T, c.L, p->S, p->Dpad, n, p->opt_chunks, c.NC_cap, p->dev.n_sm, p->dev.smem_optin, g);
}

static void fill_filter_args(const spiir_plan* p, const spiir_bank_class& c, const float* x, int n, spiir_c64* z, int accumulate,
                             const FilterGeometry& g, FilterArgs* a)
{
    a->coef = c.d_coef; a->dly = c.d_dly; a->apow = (g.scan && c.d_apow && g.C == c.apow_C) ? c.d_apow : nullptr;
    a->state = p->d_state + c.state_off; a->sstride = p->nfilt_total;
    a->chunk_st = c.d_chunk;
    a->hbuf[0] = p->d_hist[0]; a->hbuf[1] = p->d_hist[1]; a->phase = p->d_phase;
    a->x = x; a->z = reinterpret_cast<float2*>(z);
    a->n = n; a->T = c.T; a->G = c.G; a->S = p->S; a->Dpad = p->Dpad;
    a->NT = g.NT; a->CS = g.CS; a->NC = g.NC; a->C = g.C;
    a->x_aligned = ((reinterpret_cast<uintptr_t>(x) & 15u) == 0 && (p->S == 1 || (n & 3) == 0)) ? 1 : 0;
    a->accumulate = accumulate;
    a->z16 = ((reinterpret_cast<uintptr_t>(z) & 15u) == 0 && (n & 1) == 0) ? 1 : 0;
    a->mode = 0;
    a->tmap = c.d_tmap; a->T_rows = p->T; a->NP = c.NP; a->carry = 0;
}

// All classes of the plan, one after the other on the stream.  Only the very last launch writes the next input
// history and flips the ping-pong phase: every earlier launch of this call has then read the current one.
spiir_status filter_launch(spiir_plan* p, const float* x, int n, spiir_c64* z, int accumulate, cudaStream_t st)
{
    for (size_t ci = 0; ci < p->cls.size(); ++ci) {
        const spiir_bank_class& c = p->cls[ci];
        const bool last_class = ci + 1 == p->cls.size();
        FilterGeometry g;
        spiir_status rc = plan_geometry(p, c, n, &g);
        if (rc != SPIIR_OK) return rc;
        FilterArgs a;
        fill_filter_args(p, c, x, n, z, accumulate, g, &a);
        const dim3 grid(g.grid_x, g.grid_y), block(g.warps * 32);
        if (g.scan) {                                     // time-parallel scan inside one CTA per warp task: one launch
            a.carry = last_class ? 1 : 0;
            filter_kernel_t k = pick_scan_kernel(g.F, g.LPT);
            if (!k) { set_error("no scan kernel for F=%d LPT=%d", g.F, g.LPT); return SPIIR_EUNSUPPORTED; }
            SPIIR_CUDA(ensure_smem((const void*)k, g.smem_bytes));
            k<<<grid, block, g.smem_bytes, st>>>(a);
            SPIIR_CUDA(cudaGetLastError());
            continue;
        }
        for (int pass = 0; pass < (g.NC > 1 ? 2 : 1); ++pass) {
            a.mode = g.NC > 1 ? pass + 1 : 0;
            a.carry = (last_class && a.mode != 1) ? 1 : 0;
            filter_kernel_t k = pick_kernel(g.F, g.LPT, g.NP, a.mode == 1);
            if (!k) { set_error("no kernel for F=%d LPT=%d", g.F, g.LPT); return SPIIR_EUNSUPPORTED; }
            SPIIR_CUDA(ensure_smem((const void*)k, g.smem_bytes));
            k<<<grid, block, g.smem_bytes, st>>>(a);
            SPIIR_CUDA(cudaGetLastError());
            if (a.mode == 1) {
                const int nf = (int)c.nfilt;
                spiir_chunk_carry_kernel<<<(nf + 255) / 256, 256, 0, st>>>(c.d_coef, p->d_state + c.state_off, p->nfilt_total,
                                                                           c.d_chunk, nf, p->S, g.NC, g.C);
                SPIIR_CUDA(cudaGetLastError());
            }
        }
    }
    return SPIIR_OK;
}

int plan_launches(const spiir_plan* p, int n)
{
    int total = 0;
    for (const spiir_bank_class& c : p->cls) {
        FilterGeometry g;
        if (plan_geometry(p, c, n, &g) != SPIIR_OK) return 0;
        total += g.launches;
    }
    return total;
}

// Several unchunked single-class banks with the same lane mapping in ONE launch (blockIdx.z = bank).  Returns
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
        if (ps[k]->cls.size() != 1) return SPIIR_EUNSUPPORTED;
        FilterGeometry g;
        spiir_status rc = plan_geometry(ps[k], ps[k]->cls[0], ns[k], &g);
        if (rc != SPIIR_OK) return rc;
        if (g.NC != 1 || g.NP != 1) return SPIIR_EUNSUPPORTED;
        if (k == 0) { F = g.F; LPT = g.LPT; }
        else if (g.F != F || g.LPT != LPT) return SPIIR_EUNSUPPORTED;
        fill_filter_args(ps[k], ps[k]->cls[0], xs[k], ns[k], zs[k], 0, g, &m.bank[k]);
        m.bank[k].carry = 1;
        m.gx[k] = g.grid_x; m.gy[k] = g.grid_y;
        warps = std::max(warps, g.warps); gx = std::max(gx, g.grid_x); gy = std::max(gy, g.grid_y);
    }
    for (int k = 0; k < count; ++k) smem = std::max(smem, 16 * m.bank[k].CS + 16);
    multi_kernel_t k = pick_multi(F, LPT);
    if (!k) return SPIIR_EUNSUPPORTED;
    SPIIR_CUDA(ensure_smem((const void*)k, smem));
    k<<<dim3(gx, gy, count), warps * 32, smem, st>>>(m);
    SPIIR_CUDA(cudaGetLastError());
    return SPIIR_OK;
}

// ---------------------------------------------------------------------------------------------
// Device buffers of a plan, carved out of one arena.  The same code measures (arena without a base).
// ---------------------------------------------------------------------------------------------
size_t plan_layout(spiir_plan* p, Arena* a)
{
    const size_t start = a->used;
    p->d_phase = a->take_n<int>(64);
    p->d_hist[0] = a->take_n<float>((size_t)p->S * p->Dpad);
    p->d_hist[1] = a->take_n<float>((size_t)p->S * p->Dpad);
    p->d_state = a->take_n<float2>((size_t)p->S * p->nfilt_total);
    p->d_pos = a->take_n<int32_t>(p->n_filters_total);
    for (spiir_bank_class& c : p->cls) {
        c.d_coef = a->take_n<float4>(c.nfilt);
        c.d_dly = a->take_n<int32_t>(c.nfilt);
        c.d_apow = scan_mapping_supported(c.F, c.LPT, c.NP) ? a->take_n<float2>(c.nfilt) : nullptr;
        c.d_tmap = p->L_uniform ? nullptr : a->take_n<int32_t>((size_t)c.T);
        c.d_chunk = c.NC_cap > 1 ? a->take_n<float2>((size_t)c.NC_cap * p->S * c.nfilt) : nullptr;
    }
    a->used = (a->used + 255) & ~(size_t)255;
    return a->used - start;
}

// Classes of a bank: host description only (shapes, chunk capacity); arrays are filled by plan_create_in.
static spiir_status describe_classes(spiir_plan* p, const int32_t* offsets, int n_templates, int n_filters,
                                     std::vector<std::vector<int32_t>>* members)
{
    p->cls.clear();
    members->clear();
    if (!offsets) {
        spiir_bank_class c;
        c.T = n_templates; c.L = n_filters;
        if (!choose_lane_mapping(n_filters, n_templates, &c.F, &c.LPT, &c.NP)) {
            set_error("n_filters = %d not supported (1..%d)", n_filters, kMaxFiltersPerTemplate);
            return SPIIR_EUNSUPPORTED;
        }
        p->cls.push_back(c);
        members->push_back(std::vector<int32_t>());
    } else {
        // one class per lane mapping (classified as a lone template; the class's L is its longest member)
        std::map<int, int> key_to_class;
        for (int t = 0; t < n_templates; ++t) {
            const int Lt = offsets[t + 1] - offsets[t];
            int F, LPT, NP;
            if (Lt < 1 || !choose_lane_mapping(Lt, 1, &F, &LPT, &NP)) {
                set_error("template %d has %d filters (1..%d supported)", t, Lt, kMaxFiltersPerTemplate);
                return SPIIR_EUNSUPPORTED;
            }
            const int key = (F * 64 + LPT) * 16 + NP;
            auto it = key_to_class.find(key);
            if (it == key_to_class.end()) {
                spiir_bank_class c;
                c.L = 0; c.T = 0;
                it = key_to_class.emplace(key, (int)p->cls.size()).first;
                p->cls.push_back(c);
                members->push_back(std::vector<int32_t>());
            }
            (*members)[it->second].push_back(t);
            p->cls[it->second].T += 1;
            p->cls[it->second].L = std::max(p->cls[it->second].L, Lt);
        }
        // the final mapping of a class is the one of its longest member in a bank of the class's size (a large class
        // of 32..128 filters moves to half a warp per template; the places per template never shrink)
        for (spiir_bank_class& c : p->cls)
            if (!choose_lane_mapping(c.L, c.T, &c.F, &c.LPT, &c.NP)) return SPIIR_EUNSUPPORTED;
    }
    p->nfilt_total = 0;
    for (spiir_bank_class& c : p->cls) {
        c.TPG = 32 / c.LPT;
        c.G = c.LPT == 32 ? c.T * c.NP : (c.T + c.TPG - 1) / c.TPG;
        c.nfilt = (size_t)c.G * c.F * 32;
        c.state_off = p->nfilt_total;
        p->nfilt_total += c.nfilt;
        // chunk scratch: sized for the geometry of the largest block, at most 256 MiB
        c.NC_cap = 1 << 20;
        FilterGeometry g;
        spiir_status rc = plan_geometry(p, c, p->max_block, &g);
        if (rc != SPIIR_OK) return rc;
        int nc = g.scan ? 1 : g.NC;                       // the in-CTA scan keeps its chunk states in shared memory
        while (nc > 1 && (size_t)nc * p->S * c.nfilt * sizeof(float2) > ((size_t)256 << 20)) nc /= 2;
        c.NC_cap = std::max(1, nc);
    }
    return SPIIR_OK;
}

static spiir_status plan_shape(spiir_plan* p, const int32_t* offsets, int n_templates, int n_filters, int max_delay,
                               const spiir_plan_opts& o, std::vector<std::vector<int32_t>>* members)
{
    spiir_status rc = device_info(&p->dev);
    if (rc != SPIIR_OK) return rc;
    p->T = n_templates; p->S = o.n_streams; p->max_block = o.max_block;
    p->L_uniform = offsets ? 0 : n_filters;
    p->n_filters_total = offsets ? (size_t)offsets[n_templates] : (size_t)n_templates * n_filters;
    p->Dmax = max_delay; p->Dpad = std::max(4, (max_delay + 3) / 4 * 4);
    p->opt_chunks = o.time_chunks; p->flags = o.flags;
    return describe_classes(p, offsets, n_templates, n_filters, members);
}

static bool opts_ok(const spiir_plan_opts& o) { return o.n_streams >= 1 && o.max_block >= 1 && o.time_chunks >= 0; }

static bool offsets_ok(const int32_t* off, int T)
{
    if (!off || off[0] != 0) return false;
    for (int t = 0; t < T; ++t)
        if (off[t + 1] <= off[t]) return false;
    return true;
}

spiir_status plan_create_in(spiir_plan_t** out, const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays,
                            const int32_t* offsets, int n_templates, int n_filters, int rate_hz, const spiir_plan_opts& o,
                            Arena* parent)
{
    *out = nullptr;
    const size_t total = offsets ? (size_t)offsets[n_templates] : (size_t)n_templates * n_filters;
    int dmax = 0;
    for (size_t i = 0; i < total; ++i) {
        if (delays[i] < 0 || delays[i] >= (1 << 20)) { set_error("spiir_plan_create: delay out of range at %zu", i); return SPIIR_EINVAL; }
        dmax = std::max(dmax, (int)delays[i]);
    }
    spiir_plan* p = new (std::nothrow) spiir_plan;
    if (!p) return SPIIR_ENOMEM;
    p->rate_hz = rate_hz;
    std::vector<std::vector<int32_t>> members;
    spiir_status rc = plan_shape(p, offsets, n_templates, n_filters, dmax, o, &members);
    if (rc != SPIIR_OK) { delete p; return rc; }
    Arena probe;
    const size_t need = plan_layout(p, &probe);
    if (parent) {
        p->arena.base = parent->base ? static_cast<char*>(parent->take(need)) : nullptr;
        p->arena.cap = need; p->arena.owned = false;
        if (!p->arena.base) { delete p; set_error("spiir_plan_create: parent arena has no memory"); return SPIIR_ENOMEM; }
    } else {
        rc = arena_open(&p->arena, o.workspace, o.workspace_bytes, need, "spiir_plan_create");
        if (rc != SPIIR_OK) { delete p; return rc; }
    }
    plan_layout(p, &p->arena);

#define SPIIR_TRY(call)                                                                 \
    do {                                                                                \
        cudaError_t e__ = (call);                                                       \
        if (e__ != cudaSuccess) { spiir_status s__ = cuda_fail(e__, #call); spiir_plan_destroy(p); return s__; } \
    } while (0)
    std::vector<int32_t> pos(total, -1);
    for (size_t ci = 0; ci < p->cls.size(); ++ci) {
        spiir_bank_class& c = p->cls[ci];
        std::vector<float> coef;
        std::vector<int32_t> dly, cpos(total, -1);
        build_layout(a1, b0, delays, offsets, n_filters, offsets ? members[ci].data() : nullptr, c.T, c.F, c.LPT, c.NP,
                     (o.flags & 1) == 0, &coef, &dly, cpos.data());
        c.conflict_degree = layout_conflict_degree(dly, c.G, c.F);
        for (size_t i = 0; i < total; ++i)
            if (cpos[i] >= 0) pos[i] = (int32_t)(c.state_off + (size_t)cpos[i]);
        SPIIR_TRY(cudaMemcpy(c.d_coef, coef.data(), c.nfilt * sizeof(float4), cudaMemcpyHostToDevice));
        SPIIR_TRY(cudaMemcpy(c.d_dly, dly.data(), c.nfilt * sizeof(int32_t), cudaMemcpyHostToDevice));
        if (c.d_apow) {
            // chunk carry factor of the in-CTA scan at the plan's block length: a1^C in double, rounded once
            FilterGeometry g;
            c.apow_C = 0;
            if (plan_geometry(p, c, p->max_block, &g) == SPIIR_OK && g.scan) c.apow_C = g.C;
            std::vector<float> apow(c.nfilt * 2, 0.f);
            for (size_t i = 0; i < c.nfilt && c.apow_C > 0; ++i) {
                double pr = 1.0, pi = 0.0, br = (double)coef[4 * i], bi = (double)coef[4 * i + 1];
                for (int e = c.apow_C; e > 0; e >>= 1) {
                    if (e & 1) { const double r = pr * br - pi * bi, q = pr * bi + pi * br; pr = r; pi = q; }
                    const double r = br * br - bi * bi, q = 2.0 * br * bi; br = r; bi = q;
                }
                apow[2 * i] = (float)pr; apow[2 * i + 1] = (float)pi;
            }
            SPIIR_TRY(cudaMemcpy(c.d_apow, apow.data(), c.nfilt * sizeof(float2), cudaMemcpyHostToDevice));
        }
        if (c.d_tmap) SPIIR_TRY(cudaMemcpy(c.d_tmap, members[ci].data(), (size_t)c.T * sizeof(int32_t), cudaMemcpyHostToDevice));
        if (c.d_chunk) SPIIR_TRY(cudaMemset(c.d_chunk, 0, (size_t)c.NC_cap * p->S * c.nfilt * sizeof(float2)));
    }
    SPIIR_TRY(cudaMemcpy(p->d_pos, pos.data(), total * sizeof(int32_t), cudaMemcpyHostToDevice));
    SPIIR_TRY(cudaMemset(p->d_phase, 0, 64 * sizeof(int)));
    SPIIR_TRY(cudaMemset(p->d_state, 0, (size_t)p->S * p->nfilt_total * sizeof(float2)));
    SPIIR_TRY(cudaMemset(p->d_hist[0], 0, (size_t)p->S * p->Dpad * sizeof(float)));
    SPIIR_TRY(cudaMemset(p->d_hist[1], 0, (size_t)p->S * p->Dpad * sizeof(float)));
#undef SPIIR_TRY
    *out = p;
    return SPIIR_OK;
}

spiir_status plan_state_copy(spiir_plan* p, spiir_c64* y, float* hist, int to_user, cudaStream_t st)
{
    if (y) {
        const size_t TL = p->n_filters_total;
        spiir_state_permute_kernel<<<(unsigned)((TL + 255) / 256), 256, 0, st>>>(p->d_state, reinterpret_cast<float2*>(y), p->d_pos,
                                                                                 TL, p->nfilt_total, p->S, to_user);
        SPIIR_CUDA(cudaGetLastError());
    }
    if (hist || (!to_user && p->Dmax == 0)) {
        const int tot = p->S * p->Dpad;
        spiir_hist_copy_kernel<<<(tot + 255) / 256, 256, 0, st>>>(p->d_hist[0], p->d_hist[1], p->d_phase, hist, p->S, p->Dpad,
                                                                  hist ? p->Dmax : 0, to_user);
        SPIIR_CUDA(cudaGetLastError());
    }
    return SPIIR_OK;
}

}  // namespace spiir

using namespace spiir;

extern "C" {

void spiir_plan_destroy(spiir_plan_t* p)
{
    if (!p) return;
    arena_close(&p->arena);
    delete p;
}

size_t spiir_plan_workspace_bytes(int n_templates, int n_filters, int max_delay, int n_streams, int max_block, int time_chunks)
{
    if (n_templates < 1 || n_filters < 1 || max_delay < 0 || n_streams < 1 || max_block < 1 || time_chunks < 0) {
        set_error("spiir_plan_workspace_bytes: bad arguments");
        return 0;
    }
    spiir_plan p;
    std::vector<std::vector<int32_t>> members;
    spiir_plan_opts o = {n_streams, max_block, time_chunks, 0, nullptr, 0};
    if (plan_shape(&p, nullptr, n_templates, n_filters, max_delay, o, &members) != SPIIR_OK) return 0;
    Arena probe;
    return plan_layout(&p, &probe);
}

size_t spiir_plan_workspace_bytes_ragged(const int32_t* filter_offsets, int n_templates, int max_delay, int n_streams,
                                         int max_block, int time_chunks)
{
    if (n_templates < 1 || max_delay < 0 || n_streams < 1 || max_block < 1 || time_chunks < 0 || !offsets_ok(filter_offsets, n_templates)) {
        set_error("spiir_plan_workspace_bytes_ragged: bad arguments");
        return 0;
    }
    spiir_plan p;
    std::vector<std::vector<int32_t>> members;
    spiir_plan_opts o = {n_streams, max_block, time_chunks, 0, nullptr, 0};
    if (plan_shape(&p, filter_offsets, n_templates, 0, max_delay, o, &members) != SPIIR_OK) return 0;
    Arena probe;
    return plan_layout(&p, &probe);
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
    spiir_plan_opts o = {1, 4096, 0, 0, nullptr, 0};
    if (opts) o = *opts;
    if (!opts_ok(o)) { set_error("spiir_plan_create: bad options"); return SPIIR_EINVAL; }
    return plan_create_in(out, a1, b0, delays, nullptr, n_templates, n_filters, rate_hz, o, nullptr);
}

spiir_status spiir_plan_create_ragged(spiir_plan_t** out, const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays,
                                      const int32_t* filter_offsets, int n_templates, int rate_hz, const spiir_plan_opts* opts)
{
    if (!out) { set_error("spiir_plan_create_ragged: out is NULL"); return SPIIR_EINVAL; }
    *out = nullptr;
    if (!a1 || !b0 || !delays || n_templates < 1 || !offsets_ok(filter_offsets, n_templates)) {
        set_error("spiir_plan_create_ragged: NULL array, non-positive shape or offsets that do not start at 0 and increase");
        return SPIIR_EINVAL;
    }
    spiir_plan_opts o = {1, 4096, 0, 0, nullptr, 0};
    if (opts) o = *opts;
    if (!opts_ok(o)) { set_error("spiir_plan_create_ragged: bad options"); return SPIIR_EINVAL; }
    return plan_create_in(out, a1, b0, delays, filter_offsets, n_templates, 0, rate_hz, o, nullptr);
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
    SPIIR_CUDA(cudaMemsetAsync(p->d_state, 0, (size_t)p->S * p->nfilt_total * sizeof(float2), st));
    SPIIR_CUDA(cudaMemsetAsync(p->d_hist[0], 0, (size_t)p->S * p->Dpad * sizeof(float), st));
    SPIIR_CUDA(cudaMemsetAsync(p->d_hist[1], 0, (size_t)p->S * p->Dpad * sizeof(float), st));
    SPIIR_CUDA(cudaMemsetAsync(p->d_phase, 0, 2 * sizeof(int), st));
    return SPIIR_OK;
}

spiir_status spiir_plan_launch_info(const spiir_plan_t* p, int n, int info[8])
{
    if (!p || !info || n < 1) { set_error("spiir_plan_launch_info: bad arguments"); return SPIIR_EINVAL; }
    size_t big = 0;
    for (size_t ci = 1; ci < p->cls.size(); ++ci)
        if (p->cls[ci].nfilt > p->cls[big].nfilt) big = ci;
    FilterGeometry g;
    spiir_status rc = plan_geometry(p, p->cls[big], n, &g);
    if (rc != SPIIR_OK) return rc;
    info[0] = g.F; info[1] = g.LPT; info[2] = g.warps; info[3] = g.grid_x * g.grid_y;
    info[4] = g.NC; info[5] = g.smem_bytes; info[6] = g.NT; info[7] = plan_launches(p, n);
    return SPIIR_OK;
}

int spiir_plan_history_len(const spiir_plan_t* p) { return p ? p->Dmax : 0; }

spiir_status spiir_plan_get_state(spiir_plan_t* p, spiir_c64* y_out, float* hist_out, void* cuda_stream)
{
    if (!p || !y_out || (!hist_out && p->Dmax > 0)) { set_error("spiir_plan_get_state: NULL argument"); return SPIIR_EINVAL; }
    return plan_state_copy(p, y_out, hist_out, 1, static_cast<cudaStream_t>(cuda_stream));
}

spiir_status spiir_plan_set_state(spiir_plan_t* p, const spiir_c64* y_in, const float* hist_in, void* cuda_stream)
{
    if (!p || !y_in || (!hist_in && p->Dmax > 0)) { set_error("spiir_plan_set_state: NULL argument"); return SPIIR_EINVAL; }
    return plan_state_copy(p, const_cast<spiir_c64*>(y_in), const_cast<float*>(hist_in), 0, static_cast<cudaStream_t>(cuda_stream));
}

}  // extern "C"
