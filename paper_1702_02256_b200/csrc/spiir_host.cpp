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

// Filters per lane F and lanes per template LPT (power of two) with F*LPT >= L.
//   L <= 4        : one lane per template (no cross-lane sum at all)
//   5..31         : 2 / 4 / 8 lanes, 3-4 filters each
//   32..512       : the 32 lanes of a warp, F = ceil(L/32) rounded up to an instantiated F
static const int kFWarp[] = {1, 2, 3, 4, 5, 6, 7, 8, 10, 12, 14, 16};

bool choose_lane_mapping(int L, int T, int* F, int* LPT)
{
    if (L < 1) return false;
    // 32..128 filters and enough templates to give every SM several warps anyway: half a warp per template
    // (two templates per warp).  The 16 outputs of a batch then cost a 16-lane butterfly for TWO templates,
    // i.e. half the shuffle / select work per update of the one-warp-per-template mapping.
    if (L >= 32 && L <= 128 && T >= lpt16_min_templates()) { *LPT = 16; *F = (L + 15) / 16; return true; }
    if (L <= 4) { *LPT = 1; *F = L; return true; }
    if (L <= 8) { *LPT = 2; *F = (L + 1) / 2; return true; }
    if (L <= 16) { *LPT = 4; *F = (L + 3) / 4; return true; }
    if (L < 32) { *LPT = 8; *F = (L + 7) / 8; return true; }
    int need = (L + 31) / 32;
    for (int f : kFWarp)
        if (f >= need) { *LPT = 32; *F = f; return true; }
    return false;
}

int lpt16_min_templates()
{
    // measured on B200 (148 SMs): with 4096 templates the half-warp mapping is 10-30 % faster for 32..128
    // filters, with 1024 templates (3.5 warps per SM left) it is not; switch where >= 8 warps per SM remain
    return 16 * 148;
}

static inline int bank_class(int d) { return ((d + 3) >> 2) & 7; }   // 16-byte bank group of W[Dpad + j - d]

void build_layout(const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays, int T, int L, int F, int LPT,
                  bool avoid_conflicts, std::vector<float>* coef, std::vector<int32_t>* dly, std::vector<int32_t>* pos)
{
    const int TPG = 32 / LPT;
    const int G = (T + TPG - 1) / TPG;
    const size_t nf = (size_t)G * F * 32;
    coef->assign(nf * 4, 0.f);
    dly->assign(nf, 0);
    pos->assign((size_t)T * L, -1);
    std::vector<int> order;   // order[k] = filter placed at (slot, lane) position k of the template, or -1
    for (int t = 0; t < T; ++t) {
        const int32_t* d = delays + (size_t)t * L;
        order.assign((size_t)F * LPT, -1);
        if (avoid_conflicts && LPT >= 8) {
            // groups of 8 lanes (one quarter warp, one slot) should see 8 distinct bank classes
            std::vector<int> bucket[8];
            for (int l = L - 1; l >= 0; --l) bucket[bank_class(d[l])].push_back(l);
            const int ngroups = F * LPT / 8;
            int left = L;
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
                    const int f = gi / (LPT / 8), q = gi % (LPT / 8);
                    order[(size_t)f * LPT + q * 8 + r] = l;
                }
            }
        } else {
            for (int l = 0; l < L; ++l) order[(size_t)(l / LPT) * LPT + (l % LPT)] = l;
        }
        const int g = t / TPG, lane0 = (t % TPG) * LPT;
        for (int f = 0; f < F; ++f)
            for (int j = 0; j < LPT; ++j) {
                const int l = order[(size_t)f * LPT + j];
                if (l < 0) continue;
                const size_t idx = ((size_t)g * F + f) * 32 + lane0 + j;
                (*coef)[idx * 4 + 0] = a1[(size_t)t * L + l].re;
                (*coef)[idx * 4 + 1] = a1[(size_t)t * L + l].im;
                (*coef)[idx * 4 + 2] = b0[(size_t)t * L + l].re;
                (*coef)[idx * 4 + 3] = b0[(size_t)t * L + l].im;
                (*dly)[idx] = d[l];
                (*pos)[(size_t)t * L + l] = (int32_t)idx;
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

spiir_status compute_geometry(int T, int L, int S, int Dpad, int n, int opt_chunks, int nc_cap, int n_sm,
                              int smem_optin, FilterGeometry* g)
{
    memset(g, 0, sizeof *g);
    if (!choose_lane_mapping(L, T, &g->F, &g->LPT)) {
        set_error("n_filters = %d is not supported (1..512)", L);
        return SPIIR_EUNSUPPORTED;
    }
    g->TPG = 32 / g->LPT;
    g->G = (T + g->TPG - 1) / g->TPG;
    const int kBatch = 16, kMaxWarps = 8;
    // time chunks: only when the bank alone cannot fill the machine
    int NC = 1;
    const long tasks = (long)S * g->G;
    const long target = (long)n_sm * 8;
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
    // time tile: as long as shared memory allows (4 shifted copies of Dpad + NT + 32 floats)
    const int budget_floats = (smem_optin - 64) / 16;
    int NT = C;
    if (Dpad + NT + 32 > budget_floats) NT = (budget_floats - Dpad - 32) / kBatch * kBatch;
    if (NT < kBatch) {
        set_error("max delay %d does not fit the shared-memory window (limit %d samples)", Dpad, budget_floats - 48);
        return SPIIR_EUNSUPPORTED;
    }
    g->NT = NT;
    g->CS = Dpad + NT + 32;
    g->smem_bytes = 16 * g->CS + 16;
    const long W = tasks * NC;
    int warps = (int)std::min<long>(kMaxWarps, std::max<long>(1, (W + n_sm - 1) / n_sm));
    warps = std::min(warps, g->G);
    g->warps = warps;
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
const char* spiir_version(void) { return "spiir-b200 0.1 sm_100a"; }

spiir_status spiir_kaiser_taps(int n_taps, double kaiser_beta, double cutoff, float* taps_out)
{
    return spiir::kaiser_taps(n_taps, kaiser_beta, cutoff, taps_out);
}

spiir_status spiir_host_layout(const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays, int n_templates,
                               int n_filters, int avoid_conflicts, int32_t* pos_out, float* coef_out,
                               int32_t* dly_out, int info[4], double* conflict_degree)
{
    int F, LPT;
    if (!a1 || !b0 || !delays || n_templates < 1 || !spiir::choose_lane_mapping(n_filters, n_templates, &F, &LPT)) {
        spiir::set_error("spiir_host_layout: bad arguments");
        return SPIIR_EINVAL;
    }
    std::vector<float> coef;
    std::vector<int32_t> dly, pos;
    spiir::build_layout(a1, b0, delays, n_templates, n_filters, F, LPT, avoid_conflicts != 0, &coef, &dly, &pos);
    const int TPG = 32 / LPT, G = (n_templates + TPG - 1) / TPG;
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

}  // extern "C"
