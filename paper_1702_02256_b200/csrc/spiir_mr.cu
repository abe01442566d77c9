// spiir_mr.cu -- multirate SPIIR plan (Fig. 1).
//   x_0 = x, x_h = down2(x_{h-1});   z_h = bank_h(x_h);
//   acc_{H-1} = z_{H-1};  acc_{h-1} = z_{h-1} + up2(acc_h);   result acc_0 (base rate).
// Every stage keeps its own streaming history, so consecutive calls continue one stream.
#include <algorithm>
#include <stdio.h>
#include <new>
#include <vector>

#include "spiir_internal.h"

struct spiir_mr_plan {
    int H = 0, T = 0, S = 1, max_block = 0;
    std::vector<int> rates;
    std::vector<spiir_plan_t*> banks;       // [H]
    std::vector<spiir_resamp_t*> downs;     // [H-1]  x_{h} = down(x_{h-1}), rows = S
    std::vector<spiir_resamp_t*> ups;       // [H-1]  acc_{h-1} += up(acc_h), rows = S*T
    std::vector<float*> d_x;                // [H]    d_x[0] unused (caller's x)
    std::vector<spiir_c64*> d_z;            // [H]    d_z[0] unused (caller's snr_out)
    // fork / join: the H banks are independent once the down chain has run, and each of them alone is
    // too small to fill the GPU, so they are enqueued on side streams between two events
    std::vector<cudaStream_t> side;         // [H]
    std::vector<cudaEvent_t> ev_bank;       // [H]
    cudaEvent_t ev_start = nullptr, ev_chain = nullptr;
    spiir::Arena arena;                     // every device byte of the plan (caller's workspace or one library block)
};

using namespace spiir;

extern "C" {

void spiir_mr_plan_destroy(spiir_mr_plan_t* p)
{
    if (!p) return;
    for (auto b : p->banks) spiir_plan_destroy(b);
    for (auto r : p->downs) spiir_resamp_destroy(r);
    for (auto r : p->ups) spiir_resamp_destroy(r);
    for (auto q : p->side) if (q) cudaStreamDestroy(q);
    for (auto q : p->ev_bank) if (q) cudaEventDestroy(q);
    if (p->ev_start) cudaEventDestroy(p->ev_start);
    if (p->ev_chain) cudaEventDestroy(p->ev_chain);
    spiir::arena_close(&p->arena);
    delete p;
}

static const spiir_mr_opts kMrDefaults = {1, 0, 192, 5.0, 0.25, 192, 5.0, 0.25, nullptr, 0};

static bool mr_opts_ok(const spiir_mr_opts& o, int n_rates)
{
    return o.n_streams >= 1 && o.max_block >= 1 && (o.max_block % (1 << (n_rates - 1))) == 0;
}

// device bytes of a multirate plan: the banks, the stages, the per-rate strain and SNR scratch
static size_t mr_measure(int n_rates, const int* n_filters_per_rate, const int* max_delay_per_rate, int n_templates,
                         const spiir_mr_opts& o)
{
    Arena a;
    for (int h = 0; h < n_rates; ++h) {
        const int nb = o.max_block >> h;
        const size_t bank = spiir_plan_workspace_bytes(n_templates, n_filters_per_rate[h], max_delay_per_rate[h], o.n_streams, nb, 0);
        if (!bank) return 0;
        a.take(bank);
        if (h > 0) {
            const size_t dn = spiir_resamp_workspace_bytes(SPIIR_DOWN2, o.n_taps_down, o.n_streams);
            const size_t up = spiir_resamp_workspace_bytes(SPIIR_UP2, o.n_taps_up, o.n_streams * n_templates);
            if (!dn || !up) return 0;
            a.take(dn); a.take(up);
            a.take((size_t)o.n_streams * nb * sizeof(float));
            a.take((size_t)o.n_streams * n_templates * nb * sizeof(spiir_c64));
        }
    }
    return (a.used + 255) & ~(size_t)255;
}

size_t spiir_mr_workspace_bytes(int n_rates, const int* n_filters_per_rate, const int* max_delay_per_rate, int n_templates,
                                const spiir_mr_opts* opts)
{
    if (n_rates < 1 || n_rates > 16 || !n_filters_per_rate || !max_delay_per_rate || n_templates < 1 || !opts || !mr_opts_ok(*opts, n_rates)) {
        set_error("spiir_mr_workspace_bytes: bad arguments (options with max_block are required)");
        return 0;
    }
    return mr_measure(n_rates, n_filters_per_rate, max_delay_per_rate, n_templates, *opts);
}

spiir_status spiir_mr_plan_create(spiir_mr_plan_t** out, int n_rates, const int* rates_hz, const spiir_c64* const* a1,
                                  const spiir_c64* const* b0, const int32_t* const* delays,
                                  const int* n_filters_per_rate, int n_templates, const spiir_mr_opts* opts)
{
    if (!out) { set_error("spiir_mr_plan_create: out is NULL"); return SPIIR_EINVAL; }
    *out = nullptr;
    if (n_rates < 1 || n_rates > 16 || !rates_hz || !a1 || !b0 || !delays || !n_filters_per_rate || n_templates < 1) {
        set_error("spiir_mr_plan_create: bad arguments");
        return SPIIR_EINVAL;
    }
    for (int h = 1; h < n_rates; ++h)
        if (rates_hz[h] * 2 != rates_hz[h - 1]) {
            set_error("spiir_mr_plan_create: rates must halve (rate[%d] = %d, rate[%d] = %d)", h - 1, rates_hz[h - 1], h, rates_hz[h]);
            return SPIIR_EINVAL;
        }
    spiir_mr_opts o = kMrDefaults;
    o.max_block = rates_hz[0];
    if (opts) o = *opts;
    if (!mr_opts_ok(o, n_rates)) {
        set_error("spiir_mr_plan_create: max_block must be a positive multiple of 2^(n_rates-1)");
        return SPIIR_EINVAL;
    }
    std::vector<int> dmax(n_rates, 0);
    for (int h = 0; h < n_rates; ++h) {
        if (!a1[h] || !b0[h] || !delays[h] || n_filters_per_rate[h] < 1) { set_error("spiir_mr_plan_create: bad bank %d", h); return SPIIR_EINVAL; }
        const size_t TL = (size_t)n_templates * n_filters_per_rate[h];
        for (size_t i = 0; i < TL; ++i) {
            if (delays[h][i] < 0 || delays[h][i] >= (1 << 20)) { set_error("spiir_mr_plan_create: delay out of range (rate %d)", h); return SPIIR_EINVAL; }
            dmax[h] = std::max(dmax[h], (int)delays[h][i]);
        }
    }
    const size_t need = mr_measure(n_rates, n_filters_per_rate, dmax.data(), n_templates, o);
    if (!need) return SPIIR_EUNSUPPORTED;
    spiir_mr_plan* p = new (std::nothrow) spiir_mr_plan;
    if (!p) return SPIIR_ENOMEM;
    spiir_status rc = arena_open(&p->arena, o.workspace, o.workspace_bytes, need, "spiir_mr_plan_create");
    if (rc != SPIIR_OK) { delete p; return rc; }
    p->H = n_rates; p->T = n_templates; p->S = o.n_streams; p->max_block = o.max_block;
    p->rates.assign(rates_hz, rates_hz + n_rates);
    p->d_x.assign(n_rates, nullptr);
    p->d_z.assign(n_rates, nullptr);
    for (int h = 0; h < n_rates && rc == SPIIR_OK; ++h) {
        const int nb = o.max_block >> h;
        spiir_plan_opts po = {o.n_streams, nb, 0, 0, nullptr, 0};
        spiir_plan_t* b = nullptr;
        rc = plan_create_in(&b, a1[h], b0[h], delays[h], nullptr, n_templates, n_filters_per_rate[h], rates_hz[h], po, &p->arena);
        if (rc != SPIIR_OK) break;
        p->banks.push_back(b);
        if (h > 0) {
            spiir_resamp_t* d = nullptr;
            rc = resamp_create_in(&d, SPIIR_DOWN2, o.n_taps_down, o.kaiser_beta_down, o.cutoff_down, o.n_streams, nb * 2, &p->arena);
            if (rc != SPIIR_OK) break;
            p->downs.push_back(d);
            spiir_resamp_t* u = nullptr;
            rc = resamp_create_in(&u, SPIIR_UP2, o.n_taps_up, o.kaiser_beta_up, o.cutoff_up, o.n_streams * n_templates, nb, &p->arena);
            if (rc != SPIIR_OK) break;
            p->ups.push_back(u);
            p->d_x[h] = p->arena.take_n<float>((size_t)o.n_streams * nb);
            p->d_z[h] = p->arena.take_n<spiir_c64>((size_t)o.n_streams * n_templates * nb);
        }
    }
    if (rc == SPIIR_OK && n_rates > 1) {
        p->side.assign(n_rates, nullptr);
        p->ev_bank.assign(n_rates, nullptr);
        cudaError_t e = cudaEventCreateWithFlags(&p->ev_start, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_chain, cudaEventDisableTiming);
        for (int h = 0; h < n_rates && e == cudaSuccess; ++h) {
            e = cudaStreamCreateWithFlags(&p->side[h], cudaStreamNonBlocking);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_bank[h], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) rc = cuda_fail(e, "spiir_mr_plan_create streams");
    }
    if (rc != SPIIR_OK) { spiir_mr_plan_destroy(p); return rc; }
    *out = p;
    return SPIIR_OK;
}

spiir_status spiir_mr_filter(spiir_mr_plan_t* p, const float* x, int n, spiir_c64* snr_out, void* cuda_stream)
{
    if (!p || n < 0) { set_error("spiir_mr_filter: bad plan or n"); return SPIIR_EINVAL; }
    if (n == 0) return SPIIR_OK;
    if (!x || !snr_out) { set_error("spiir_mr_filter: NULL buffer"); return SPIIR_EINVAL; }
    if (n % (1 << (p->H - 1)) != 0) { set_error("spiir_mr_filter: n = %d is not a multiple of 2^(H-1) = %d", n, 1 << (p->H - 1)); return SPIIR_EINVAL; }
    if (n > p->max_block) { set_error("spiir_mr_filter: n exceeds max_block"); return SPIIR_ESTATE; }
    if (reinterpret_cast<uintptr_t>(snr_out) & 15u) { set_error("spiir_mr_filter: snr_out must be 16-byte aligned"); return SPIIR_EINVAL; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    spiir_status rc;
    if (p->H == 1) return filter_launch(p->banks[0], x, n, snr_out, 0, st);
    // fork: the base-rate bank needs only x
    SPIIR_CUDA(cudaEventRecord(p->ev_start, st));
    SPIIR_CUDA(cudaStreamWaitEvent(p->side[0], p->ev_start, 0));
    rc = filter_launch(p->banks[0], x, n, snr_out, 0, p->side[0]);
    if (rc != SPIIR_OK) return rc;
    SPIIR_CUDA(cudaEventRecord(p->ev_bank[0], p->side[0]));
    // row a8: down chain, one launch (falls back to one launch per stage for other tap counts)
    rc = down_chain_launch(p->downs.data(), p->H - 1, x, n, p->d_x.data() + 1, p->S, st);
    if (rc == SPIIR_EUNSUPPORTED) {
        const float* xh = x;
        for (int h = 1; h < p->H; ++h) {
            rc = spiir_resample_down(p->downs[h - 1], xh, n >> (h - 1), p->d_x[h], st);
            if (rc != SPIIR_OK) return rc;
            xh = p->d_x[h];
        }
    } else if (rc != SPIIR_OK) return rc;
    SPIIR_CUDA(cudaEventRecord(p->ev_chain, st));
    // row a9: per-rate banks, side by side.  Unchunked banks that share a lane mapping go out as ONE launch
    // (the low rates are a few microseconds of work each); everything else gets its own side stream.
    std::vector<char> done(p->H, 0), rec(p->H, 0);
    rec[0] = 1;
    for (int h = 1; h < p->H; ++h) {
        if (done[h]) continue;
        FilterGeometry gh;
        if ((rc = plan_geometry(p->banks[h], p->banks[h]->cls[0], n >> h, &gh)) != SPIIR_OK) return rc;
        std::vector<int> grp(1, h);
        if (gh.NC == 1 && gh.NP == 1)
            for (int j = h + 1; j < p->H && (int)grp.size() < 8; ++j) {
                FilterGeometry gj;
                if (done[j] || plan_geometry(p->banks[j], p->banks[j]->cls[0], n >> j, &gj) != SPIIR_OK) continue;
                if (gj.NC == 1 && gj.NP == 1 && gj.F == gh.F && gj.LPT == gh.LPT) grp.push_back(j);
            }
        SPIIR_CUDA(cudaStreamWaitEvent(p->side[h], p->ev_chain, 0));
        rc = SPIIR_EUNSUPPORTED;
        if (grp.size() >= 2) {
            spiir_plan* ps[8]; const float* xs[8]; int ns[8]; spiir_c64* zs[8];
            for (size_t k = 0; k < grp.size(); ++k) { ps[k] = p->banks[grp[k]]; xs[k] = p->d_x[grp[k]]; ns[k] = n >> grp[k]; zs[k] = p->d_z[grp[k]]; }
            rc = filter_launch_group(ps, xs, ns, zs, (int)grp.size(), p->side[h]);
            if (rc == SPIIR_OK) for (int j : grp) done[j] = 1;
            else if (rc != SPIIR_EUNSUPPORTED) return rc;
        }
        if (rc == SPIIR_EUNSUPPORTED) {
            rc = filter_launch(p->banks[h], p->d_x[h], n >> h, p->d_z[h], 0, p->side[h]);
            if (rc != SPIIR_OK) return rc;
            done[h] = 1;
        }
        SPIIR_CUDA(cudaEventRecord(p->ev_bank[h], p->side[h]));
        rec[h] = 1;
    }
    for (int h = 0; h < p->H; ++h)                                                         // join
        if (rec[h]) SPIIR_CUDA(cudaStreamWaitEvent(st, p->ev_bank[h], 0));
    // row a10: up + accumulate cascade, lowest rate first; one launch when the tap count has a fused kernel
    {
        const int nst = p->H - 1;
        std::vector<spiir_resamp*> ups(nst);
        std::vector<const spiir_c64*> zadd(nst);
        for (int k = 0; k < nst; ++k) {
            const int h = p->H - 1 - k;                   // stage k lifts rate h to rate h-1
            ups[k] = p->ups[h - 1];
            zadd[k] = h == 1 ? snr_out : p->d_z[h - 1];
        }
        rc = up_chain_launch(ups.data(), nst, p->d_z[p->H - 1], n >> (p->H - 1), zadd.data(), snr_out, p->S * p->T, st);
        if (rc == SPIIR_EUNSUPPORTED) {
            for (int h = p->H - 1; h >= 1; --h) {
                rc = spiir_resample_up(p->ups[h - 1], p->d_z[h], n >> h, h == 1 ? snr_out : p->d_z[h - 1], 1, st);
                if (rc != SPIIR_OK) return rc;
            }
        } else if (rc != SPIIR_OK) return rc;
    }
    return SPIIR_OK;
}

spiir_status spiir_mr_plan_reset(spiir_mr_plan_t* p, void* cuda_stream)
{
    if (!p) { set_error("spiir_mr_plan_reset: NULL plan"); return SPIIR_EINVAL; }
    spiir_status rc = SPIIR_OK;
    for (auto b : p->banks) if ((rc = spiir_plan_reset(b, cuda_stream)) != SPIIR_OK) return rc;
    for (auto r : p->downs) if ((rc = spiir_resamp_reset(r, cuda_stream)) != SPIIR_OK) return rc;
    for (auto r : p->ups) if ((rc = spiir_resamp_reset(r, cuda_stream)) != SPIIR_OK) return rc;
    return rc;
}

// Resume state blob (layout in include/spiir.h): sections in a fixed order, each 16-byte aligned.
static size_t mr_state_walk(spiir_mr_plan_t* p, char* blob, int to_user, cudaStream_t st, spiir_status* rc)
{
    size_t off = 0;
    auto section = [&](size_t bytes) { const size_t at = off; off = (off + bytes + 15) & ~(size_t)15; return at; };
    *rc = SPIIR_OK;
    for (int h = 0; h < p->H && *rc == SPIIR_OK; ++h) {
        spiir_plan* b = p->banks[h];
        const size_t ay = section((size_t)b->S * b->n_filters_total * sizeof(spiir_c64));
        const size_t ah = section((size_t)b->S * b->Dmax * sizeof(float));
        if (blob) *rc = plan_state_copy(b, reinterpret_cast<spiir_c64*>(blob + ay), b->Dmax ? reinterpret_cast<float*>(blob + ah) : nullptr,
                                        to_user, st);
    }
    for (size_t k = 0; k < p->downs.size() && *rc == SPIIR_OK; ++k) {
        const size_t at = section((size_t)p->downs[k]->rows * p->downs[k]->H * sizeof(float));
        if (blob) *rc = resamp_state_copy(p->downs[k], blob + at, to_user, st);
    }
    for (size_t k = 0; k < p->ups.size() && *rc == SPIIR_OK; ++k) {
        const size_t at = section((size_t)p->ups[k]->rows * p->ups[k]->H * sizeof(spiir_c64));
        if (blob) *rc = resamp_state_copy(p->ups[k], blob + at, to_user, st);
    }
    return off;
}

size_t spiir_mr_plan_state_bytes(const spiir_mr_plan_t* p)
{
    if (!p) return 0;
    spiir_status rc;
    return mr_state_walk(const_cast<spiir_mr_plan_t*>(p), nullptr, 1, nullptr, &rc);
}

spiir_status spiir_mr_plan_get_state(spiir_mr_plan_t* p, void* blob_out, void* cuda_stream)
{
    if (!p || !blob_out || (reinterpret_cast<uintptr_t>(blob_out) & 15u)) { set_error("spiir_mr_plan_get_state: NULL or misaligned blob"); return SPIIR_EINVAL; }
    spiir_status rc;
    mr_state_walk(p, static_cast<char*>(blob_out), 1, static_cast<cudaStream_t>(cuda_stream), &rc);
    return rc;
}

spiir_status spiir_mr_plan_set_state(spiir_mr_plan_t* p, const void* blob_in, void* cuda_stream)
{
    if (!p || !blob_in || (reinterpret_cast<uintptr_t>(blob_in) & 15u)) { set_error("spiir_mr_plan_set_state: NULL or misaligned blob"); return SPIIR_EINVAL; }
    spiir_status rc;
    mr_state_walk(p, static_cast<char*>(const_cast<void*>(blob_in)), 0, static_cast<cudaStream_t>(cuda_stream), &rc);
    return rc;
}

int spiir_mr_launches(const spiir_mr_plan_t* p, int n)
{
    if (!p || n < 1) return 0;
    int total = 0;
    if (p->H > 1) {
        // fused down chain / fused up cascade when they apply (tap count, shared memory), else one launch per stage
        total += down_chain_fits(p->downs.data(), p->H - 1, n) ? 1 : p->H - 1;
        std::vector<spiir_resamp*> ups(p->H - 1);
        for (int k = 0; k < p->H - 1; ++k) ups[k] = p->ups[p->H - 2 - k];
        total += up_chain_fits(ups.data(), p->H - 1, n >> (p->H - 1)) ? 1 : p->H - 1;
    }
    std::vector<FilterGeometry> g(p->H);
    for (int h = 0; h < p->H; ++h)
        if (plan_geometry(p->banks[h], p->banks[h]->cls[0], std::max(1, n >> h), &g[h]) != SPIIR_OK) return 0;
    std::vector<char> done(p->H, 0);
    for (int h = 0; h < p->H; ++h) {
        if (done[h]) continue;
        total += plan_launches(p->banks[h], std::max(1, n >> h));
        done[h] = 1;
        // the same grouping as spiir_mr_filter: unchunked banks h >= 1 with one warp per template and F <= 8
        if (h >= 1 && g[h].NC == 1 && g[h].NP == 1 && g[h].LPT == 32 && g[h].F <= 8) {
            int members = 1;
            for (int j = h + 1; j < p->H && members < 8; ++j)
                if (!done[j] && g[j].NC == 1 && g[j].NP == 1 && g[j].F == g[h].F && g[j].LPT == g[h].LPT) { done[j] = 1; ++members; }
        }
    }
    return total;
}

}  // extern "C"
