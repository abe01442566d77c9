// spiir_host.cpp -- host-only logic of libspiir.so: error text, lane mapping, bank-conflict-aware
// filter permutation, launch geometry, Kaiser taps.  Nothing here touches the GPU, so it is
// covered by the CPU test-suite through the spiir_host_* entry points.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>

#include "spiir_internal.h"

namespace spiir {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}

const char* last_error() { return g_err; }

// Filters per lane F, lanes per template LPT (power of two) and warps per template NP with F*LPT*NP >= L.
//   L <= 4        : one lane per template (no cross-lane sum at all)
//   5..31         : 2 / 4 / 8 lanes, 3-4 filters each
//   32..64, 65..128 in a bank of >= 2368 templates: 8 lanes (4..8 filters each), 16 lanes (5..8 filters each)
//   32..512       : the 32 lanes of a warp, F = ceil(L/32) rounded up to an instantiated F
//   513..2048     : NP = 2..8 adjacent warps of one CTA, F <= 8 each (a 513-filter template takes 544
//                   threads of one block); the pair (NP, F) with the least padding wins, fewer warps on a tie
static const int kFWarp[] = {1, 2, 3, 4, 5, 6, 7, 8, 10, 12, 14, 16};

bool choose_lane_mapping(int L, int T, int* F, int* LPT, int* NP)
{
    *NP = 1;
    if (L < 1 || L > kMaxFiltersPerTemplate) return false;
    // 32..128 filters and enough templates to give every SM several warps anyway: half a warp per template
    // (two templates per warp).  The 16 outputs of a batch then cost a 16-lane butterfly for TWO templates,
    // i.e. half the shuffle / select work per update of the one-warp-per-template mapping.
    // 32..64 filters in such a bank: a quarter warp per template (four templates per warp, 4..8 filters per lane).  Measured
    // against the half-warp mapping on 4096 templates: 256-sample blocks 7 % (L = 32), 5 % (48), 0 % (64) faster, one call
    // of 16384 samples 24 %, 22 %, 17 % faster (an 8-lane butterfly per 4..8 filters instead of a 16-lane one per 2..4).
    if (L >= 32 && L <= 64 && T >= lpt16_min_templates()) { *LPT = 8; *F = (L + 7) / 8; return true; }
    if (L >= 32 && L <= 128 && T >= lpt16_min_templates()) { *LPT = 16; *F = (L + 15) / 16; return true; }
    if (L < 32) {
        if (L <= 4) { *LPT = 1; *F = L; }
        else if (L <= 8) { *LPT = 2; *F = (L + 1) / 2; }
        else if (L <= 16) { *LPT = 4; *F = (L + 3) / 4; }
        else { *LPT = 8; *F = (L + 7) / 8; }
        // A mid-sized bank of very short templates gives too few warp tasks (= CTAs of the in-CTA time scan) to cover the
        // SMs: 1024 templates x 8 filters at 2 lanes each are 64 tasks on 148 SMs.  Twice the lanes per template doubles
        // the tasks; the extra butterfly stage costs less than the idle SMs (configs[3] base rate: 69 -> 40 us).
        while (T >= 512 && *LPT < 8 && *F >= 4 && (long)((T * *LPT + 31) / 32) * 4 < 3L * 148) {
            *LPT *= 2;
            *F = (L + *LPT - 1) / *LPT;
        }
        return true;
    }
    *LPT = 32;
    if (L <= 512) {
        const int need = (L + 31) / 32;
        for (int f : kFWarp)
            if (f >= need) { *F = f; return true; }
        return false;
    }
    int best = 1 << 30;
    for (int np = 2; np <= 8; ++np) {
        const int f = (L + 32 * np - 1) / (32 * np);
        if (f > 8) continue;
        if (f * 32 * np < best) { best = f * 32 * np; *F = f; *NP = np; }
    }
    return best < (1 << 30);
}

int lpt16_min_templates()
{
    // measured on B200 (148 SMs): with 4096 templates the half-warp mapping is 10-30 % faster for 32..128
    // filters, with 1024 templates (3.5 warps per SM left) it is not; switch where >= 8 warps per SM remain
    return 16 * 148;
}

static inline int bank_class(int d) { return ((d + 3) >> 2) & 7; }   // 16-byte bank group of W[Dpad + j - d]

void build_layout(const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays, const int32_t* offsets, int L,
                  const int32_t* templates, int T, int F, int LPT, int NP, bool avoid_conflicts,
                  std::vector<float>* coef, std::vector<int32_t>* dly, int32_t* pos)
{
    const int TPG = 32 / LPT;
    const int G = LPT == 32 ? T * NP : (T + TPG - 1) / TPG;
    const size_t nf = (size_t)G * F * 32;
    const int slots = NP * F * LPT;                        // filter places of one template
    coef->assign(nf * 4, 0.f);
    dly->assign(nf, 0);
    std::vector<int> order;   // order[k] = filter (index within the template) placed at place k = (piece, slot, lane), or -1
    for (int tc = 0; tc < T; ++tc) {
        const int t = templates ? templates[tc] : tc;
        const size_t base = offsets ? (size_t)offsets[t] : (size_t)t * L;
        const int Lt = offsets ? offsets[t + 1] - offsets[t] : L;
        const int32_t* d = delays + base;
        order.assign((size_t)slots, -1);
        if (avoid_conflicts && LPT >= 8) {
            // groups of 8 lanes (one quarter warp, one slot) should see 8 distinct bank classes
            std::vector<int> bucket[8];
            for (int l = Lt - 1; l >= 0; --l) bucket[bank_class(d[l])].push_back(l);
            const int ngroups = slots / 8;
            int left = Lt;
            for (int gi = 0; gi < ngroups && left > 0; ++gi) {
                bool used[8] = {false, false, false, false, false, false, false, false};
                for (int r = 0; r < 8 && left > 0; ++r) {
                    int best = -1;
                    for (int c = 0; c < 8; ++c)
                        if (!used[c] && !bucket[c].empty() && (best < 0 || bucket[c].size() > bucket[best].size())) best = c;
                    if (best < 0)
                        for (int c = 0; c < 8; ++c)
                            if (!bucket[c].empty() && (best < 0 || bucket[c].size() > bucket[best].size())) best = c;
                    used[best] = true;
                    const int l = bucket[best].back();
                    bucket[best].pop_back();
                    --left;
                    order[(size_t)gi * 8 + r] = l;         // place = (piece, slot, quarter) * 8 + r: slot-major inside a piece
                }
            }
        } else {
            for (int l = 0; l < Lt; ++l) order[(size_t)l] = l;
        }
        for (int k = 0; k < slots; ++k) {
            const int l = order[(size_t)k];
            if (l < 0) continue;
            const int piece = k / (F * LPT), f = (k % (F * LPT)) / LPT, j = k % LPT;
            const int g = LPT == 32 ? tc * NP + piece : tc / TPG;
            const int lane0 = LPT == 32 ? 0 : (tc % TPG) * LPT;
            const size_t idx = ((size_t)g * F + f) * 32 + lane0 + j;
            (*coef)[idx * 4 + 0] = a1[base + l].re;
            (*coef)[idx * 4 + 1] = a1[base + l].im;
            (*coef)[idx * 4 + 2] = b0[base + l].re;
            (*coef)[idx * 4 + 3] = b0[base + l].im;
            (*dly)[idx] = d[l];
            if (pos) pos[base + l] = (int32_t)idx;
        }
    }
}

double layout_conflict_degree(const std::vector<int32_t>& dly, int G, int F)
{
    double total = 0.0;
    size_t cnt = 0;
    for (int g = 0; g < G; ++g)
        for (int f = 0; f < F; ++f)
            for (int q = 0; q < 4; ++q) {
                int hist[8] = {0, 0, 0, 0, 0, 0, 0, 0};
                int worst = 0;
                for (int r = 0; r < 8; ++r) {
                    int c = bank_class(dly[((size_t)g * F + f) * 32 + q * 8 + r]);
                    worst = std::max(worst, ++hist[c]);
                }
                total += worst;
                ++cnt;
            }
    return cnt ? total / (double)cnt : 0.0;
}

// ---------------------------------------------------------------------------------------------
// Launch geometry.  Pure function of the bank shape, the block length and the device limits.
// ---------------------------------------------------------------------------------------------
static inline int round_up(int v, int m) { return (v + m - 1) / m * m; }

bool scan_mapping_supported(int F, int LPT, int NP) { return NP == 1 && F <= 4 && LPT <= 8; }

spiir_status compute_geometry(int T, int L, int S, int Dpad, int n, int opt_chunks, int nc_cap, int n_sm,
                              int smem_optin, FilterGeometry* g)
{
    memset(g, 0, sizeof *g);
    if (!choose_lane_mapping(L, T, &g->F, &g->LPT, &g->NP)) {
        set_error("n_filters = %d is not supported (1..%d)", L, kMaxFiltersPerTemplate);
        return SPIIR_EUNSUPPORTED;
    }
    g->TPG = 32 / g->LPT;
    g->G = g->LPT == 32 ? T * g->NP : (T + g->TPG - 1) / g->TPG;
    const int kBatch = 16, kMaxWarps = 8, kScanMaxWarps = 16;
    const int kTileRowBytes = 9 * 16;                      // spiir_filter.cuh: kTileRow4 float4 per store-tile row
    const int kRedWarpBytes = (32 * 9 + 64) * 16;          // spiir_filter.cuh: kRedWarp4 float4 per warp (multi-warp templates)
    // time chunks: only when the bank alone cannot fill the machine
    int NC = 1;
    const long tasks = (long)S * g->G;
    const long target = (long)n_sm * 8;
    // Few filters per template (several templates per warp, F <= 4): the chunks are the warps of one CTA per warp
    // task and the carry goes through shared memory -- one launch, so it pays for blocks as short as 64 samples.
    if (scan_mapping_supported(g->F, g->LPT, g->NP) && opt_chunks != 1 && n >= 64) {
        long ncw = opt_chunks > 1 ? opt_chunks : (tasks * 2 <= target ? 2 * target / tasks : 1);
        ncw = std::min<long>(std::min<long>(ncw, kScanMaxWarps), n / 32);
        if (ncw >= 2) {
            const int ex_bytes = ((int)ncw + 1) * g->F * 32 * 8 + (g->LPT <= 4 ? (int)ncw * g->TPG * kTileRowBytes : 0);   // chunk states + store tiles
            const int budget = (smem_optin - 64 - ex_bytes) / 16;
            int NT = round_up(n, kBatch);
            if (Dpad + NT + 32 > budget) {                 // several time tiles of equal length
                const int nt_max = (budget - Dpad - 32) / kBatch * kBatch;
                const int ntiles = nt_max >= 64 ? (n + nt_max - 1) / nt_max : 0;
                NT = ntiles ? round_up((n + ntiles - 1) / ntiles, kBatch) : 0;
            }
            if (NT >= 64) {
                const int C = round_up((NT + (int)ncw - 1) / (int)ncw, kBatch);
                g->scan = 1; g->NC = (NT + C - 1) / C; g->C = C; g->NT = NT; g->CS = Dpad + NT + 32;
                g->warps = g->NC; g->grid_x = g->G; g->grid_y = S; g->launches = 1;
                g->smem_bytes = 16 * g->CS + 16 + ex_bytes;
                return SPIIR_OK;
            }
        }
    }
    if (opt_chunks >= 1) NC = opt_chunks;
    else if (tasks * 2 <= target && n >= 128) {
        // Chunking costs two more launches and 1.75x the arithmetic; it pays only when the time a lone
        // warp needs for the whole block exceeds that.  Cost model from measurements on B200: ~8 us per
        // launch (window staging, coefficient loads, tail), ~36 ns per time step of a warp, and
        // proportionally more once more than 4 warps share an SM.
        const long nc = std::min<long>(target / tasks, n / 64);
        if (nc >= 2) {
            const double f0 = 8e-6, tau = 36e-9;
            const double share_p = std::max(1.0, (double)((tasks + n_sm - 1) / n_sm) / 4.0);
            const double share_c = std::max(1.0, (double)((tasks * nc + n_sm - 1) / n_sm) / 4.0);
            const double t_plain = f0 + n * tau * share_p;
            const double t_chunk = 3.0 * f0 + ((double)n / (double)nc) * tau * 1.75 * share_c;
            if (t_chunk * 1.15 < t_plain) NC = (int)nc;
        }
    }
    NC = std::max(1, std::min(NC, nc_cap));
    int C = round_up((n + NC - 1) / NC, kBatch);
    NC = (n + C - 1) / C;
    if (NC <= 1) { NC = 1; C = round_up(std::max(n, 1), kBatch); }
    g->NC = NC; g->C = C;
    const long W = tasks * NC;
    int warps = (int)std::min<long>(kMaxWarps, std::max<long>(1, (W + n_sm - 1) / n_sm));
    warps = std::min(warps, g->G);
    if (g->NP > 1) warps = std::max(g->NP, warps / g->NP * g->NP);      // the warps of a template share a CTA
    g->warps = warps;
    const int red_bytes = g->NP > 1 ? warps * kRedWarpBytes : (g->LPT <= 4 ? warps * g->TPG * kTileRowBytes : 0);   // or the store tiles
    // time tile: as long as shared memory allows (4 shifted copies of Dpad + NT + 32 floats)
    const int budget_floats = (smem_optin - 64 - red_bytes) / 16;
    int NT = C;
    if (Dpad + NT + 32 > budget_floats) NT = (budget_floats - Dpad - 32) / kBatch * kBatch;
    if (NT < kBatch) {
        set_error("max delay %d does not fit the shared-memory window (limit %d samples)", Dpad, budget_floats - 48);
        return SPIIR_EUNSUPPORTED;
    }
    g->NT = NT;
    g->CS = Dpad + NT + 32;
    g->smem_bytes = 16 * g->CS + 16 + red_bytes;
    int gx = (g->G + warps - 1) / warps;
    const int resident = std::max(1, (2 * n_sm) / (S * NC));   // CTAs per (stream, chunk) kept resident
    if (gx > resident && (long)gx * S * NC > 2L * n_sm) gx = resident;
    g->grid_x = gx;
    g->grid_y = S * NC;
    g->launches = NC > 1 ? 3 : 1;
    return SPIIR_OK;
}

// ---------------------------------------------------------------------------------------------
// Kaiser-windowed sinc (Eq. 9; readings R1-R3).  I0 by its power series with the
// terms generated from the ratio of consecutive terms.
// ---------------------------------------------------------------------------------------------
static double i0_series(double v)
{
    const double q = 0.25 * v * v;
    double term = 1.0, sum = 1.0;
    for (int k = 1; k < 1000; ++k) {
        term *= q / ((double)k * (double)k);
        sum += term;
        if (term < sum * 1e-18) break;
    }
    return sum;
}

spiir_status kaiser_taps(int n_taps, double beta, double cutoff, float* out)
{
    if (!out || n_taps < 2 || n_taps > 1024 || !(cutoff > 0.0) || !(cutoff <= 0.5) || !(beta >= 0.0)) {
        set_error("spiir_kaiser_taps: bad arguments");
        return SPIIR_EINVAL;
    }
    std::vector<double> h(n_taps);
    const double mid = 0.5 * (n_taps - 1), inv_i0b = 1.0 / i0_series(beta);
    double total = 0.0;
    for (int j = 0; j < n_taps; ++j) {
        const double u = (j - mid) / mid;                       // -1 .. 1
        const double win = i0_series(beta * sqrt(std::max(0.0, 1.0 - u * u))) * inv_i0b;
        const double arg = M_PI * 2.0 * cutoff * (j - mid);
        const double lp = (fabs(arg) < 1e-300) ? 2.0 * cutoff : 2.0 * cutoff * sin(arg) / arg;
        h[j] = win * lp;
        total += h[j];
    }
    for (int j = 0; j < n_taps; ++j) out[j] = (float)(h[j] / total);
    return SPIIR_OK;
}

}  // namespace spiir

extern "C" {

const char* spiir_last_error(void) { return spiir::last_error(); }
const char* spiir_version(void) { return "spiir-b200 0.2 sm_100a"; }

spiir_status spiir_kaiser_taps(int n_taps, double kaiser_beta, double cutoff, float* taps_out)
{
    return spiir::kaiser_taps(n_taps, kaiser_beta, cutoff, taps_out);
}

spiir_status spiir_host_layout(const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays, int n_templates,
                               int n_filters, int avoid_conflicts, int32_t* pos_out, float* coef_out,
                               int32_t* dly_out, int info[4], double* conflict_degree)
{
    int F, LPT, NP;
    if (!a1 || !b0 || !delays || n_templates < 1 || !spiir::choose_lane_mapping(n_filters, n_templates, &F, &LPT, &NP)) {
        spiir::set_error("spiir_host_layout: bad arguments");
        return SPIIR_EINVAL;
    }
    std::vector<float> coef;
    std::vector<int32_t> dly, pos((size_t)n_templates * n_filters, -1);
    spiir::build_layout(a1, b0, delays, nullptr, n_filters, nullptr, n_templates, F, LPT, NP, avoid_conflicts != 0, &coef, &dly,
                        pos.data());
    const int TPG = 32 / LPT, G = LPT == 32 ? n_templates * NP : (n_templates + TPG - 1) / TPG;
    if (info) { info[0] = F; info[1] = LPT; info[2] = G; info[3] = (int)(dly.size()); }
    if (pos_out) memcpy(pos_out, pos.data(), pos.size() * sizeof(int32_t));
    if (coef_out) memcpy(coef_out, coef.data(), coef.size() * sizeof(float));
    if (dly_out) memcpy(dly_out, dly.data(), dly.size() * sizeof(int32_t));
    if (conflict_degree) *conflict_degree = spiir::layout_conflict_degree(dly, G, F);
    return SPIIR_OK;
}

spiir_status spiir_host_geometry(int n_templates, int n_filters, int n_streams, int max_delay, int n,
                                 int time_chunks, int n_sm, int smem_optin, int info[8])
{
    if (n_templates < 1 || n_streams < 1 || max_delay < 0 || n < 1 || n_sm < 1 || !info) {
        spiir::set_error("spiir_host_geometry: bad arguments");
        return SPIIR_EINVAL;
    }
    spiir::FilterGeometry g;
    const int Dpad = (max_delay + 3) / 4 * 4;
    spiir_status st = spiir::compute_geometry(n_templates, n_filters, n_streams, Dpad, n, time_chunks, 1 << 20, n_sm,
                                              smem_optin, &g);
    if (st != SPIIR_OK) return st;
    info[0] = g.F; info[1] = g.LPT; info[2] = g.warps; info[3] = g.grid_x * g.grid_y;
    info[4] = g.NC; info[5] = g.smem_bytes; info[6] = g.NT; info[7] = g.launches;
    return SPIIR_OK;
}

spiir_status spiir_host_lane_mapping(int n_filters, int n_templates, int info[3])
{
    int F, LPT, NP;
    if (!info || n_templates < 1 || !spiir::choose_lane_mapping(n_filters, n_templates, &F, &LPT, &NP)) {
        spiir::set_error("spiir_host_lane_mapping: n_filters = %d not supported (1..%d)", n_filters, spiir::kMaxFiltersPerTemplate);
        return SPIIR_EUNSUPPORTED;
    }
    info[0] = F; info[1] = LPT; info[2] = NP;
    return SPIIR_OK;
}

// PAPER.md:79, reading R8 (see include/spiir.h).
spiir_status spiir_assign_rates(const spiir_c64* a1, int n, int base_rate_hz, const int* rates_hz, int n_rates,
                                double band_factor, int32_t* rate_index_out)
{
    if (!a1 || !rates_hz || !rate_index_out || n < 0 || n_rates < 1 || base_rate_hz < 1 || rates_hz[0] != base_rate_hz ||
        !(band_factor >= 0.0)) {
        spiir::set_error("spiir_assign_rates: bad arguments");
        return SPIIR_EINVAL;
    }
    for (int h = 1; h < n_rates; ++h)
        if (rates_hz[h] >= rates_hz[h - 1] || rates_hz[h] < 1) { spiir::set_error("spiir_assign_rates: rates must descend"); return SPIIR_EINVAL; }
    for (int i = 0; i < n; ++i) {
        const double re = a1[i].re, im = a1[i].im, mag = hypot(re, im);
        int pick = 0;
        if (mag > 0.0 && mag < 1.0) {
            const double f0 = fabs(atan2(im, re)) * base_rate_hz / (2.0 * M_PI);
            const double df = -log(mag) * base_rate_hz / (2.0 * M_PI);
            const double nyq = 2.0 * (f0 + band_factor * df);
            for (int h = n_rates - 1; h >= 0; --h)
                if ((double)rates_hz[h] >= nyq) { pick = h; break; }     // lowest available rate that still holds the band
        }
        rate_index_out[i] = pick;
    }
    return SPIIR_OK;
}

}  // extern "C"
