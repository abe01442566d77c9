// spiir_internal.h -- host-side structures shared by the translation units of libspiir.so.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/spiir.h"

namespace spiir {

void set_error(const char* fmt, ...);
spiir_status cuda_fail(cudaError_t e, const char* what);

#define SPIIR_CUDA(call)                                             \
    do {                                                             \
        cudaError_t e__ = (call);                                    \
        if (e__ != cudaSuccess) return spiir::cuda_fail(e__, #call); \
    } while (0)

struct DeviceInfo {
    int device = -1;
    int n_sm = 0;
    int smem_optin = 0;   // max dynamic shared memory per block (opt-in)
};
spiir_status device_info(DeviceInfo* out);
cudaError_t ensure_smem(const void* func, int bytes);

// Bump allocator over ONE device block: the caller's workspace, or a block the library allocated itself.
// With base == nullptr it only measures (the *_workspace_bytes entry points run the same layout code).
struct Arena {
    char* base = nullptr;
    size_t cap = 0, used = 0;
    bool owned = false;               // base came from cudaMalloc and is freed with the plan
    bool measuring() const { return base == nullptr; }
    void* take(size_t bytes)
    {
        const size_t off = (used + 255) & ~(size_t)255;
        used = off + bytes;
        return base ? base + off : nullptr;
    }
    template <typename T> T* take_n(size_t n) { return static_cast<T*>(take(n * sizeof(T))); }
};
// opts workspace -> arena (checks alignment and size against `need`), or one cudaMalloc of `need` bytes
spiir_status arena_open(Arena* a, void* workspace, size_t workspace_bytes, size_t need, const char* who);
void arena_close(Arena* a);

// Launch geometry of the filter kernel for one block length (host logic, testable without a GPU).
struct FilterGeometry {
    int F, LPT, TPG, NP, G;   // filters per lane, lanes per template, templates per group, warps per template, warp tasks
    int NC, C;                // time chunks and chunk length
    int NT, CS;               // time tile and shifted-copy stride (floats)
    int warps, grid_x, grid_y;
    int smem_bytes;
    int launches;
    int scan;                 // NC chunks are the warps of ONE CTA per warp task (spiir_filter_scan_kernel), one launch
};

constexpr int kMaxFiltersPerTemplate = 2048;

// Pick (F, LPT, NP) for a bank of L filters per template.  Returns false when L is not supported.
bool choose_lane_mapping(int L, int T, int* F, int* LPT, int* NP);
int lpt16_min_templates();
bool scan_mapping_supported(int F, int LPT, int NP);   // spiir_filter_scan_kernel is instantiated for this mapping

// One class of a plan: fills the permuted coefficient / delay arrays ([G][F][32], zero padded) and, for every filter of
// the listed templates, its index in them.  offsets == nullptr: uniform bank of L filters per template (template t owns
// [t*L, (t+1)*L)); else CSR offsets.  templates: ids of the class's templates in class order (nullptr: 0..T-1).
// pos (flat filter index -> plan index) is written only for the listed templates.
void build_layout(const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays, const int32_t* offsets, int L,
                  const int32_t* templates, int T, int F, int LPT, int NP, bool avoid_conflicts,
                  std::vector<float>* coef /* [G*F*32*4] */, std::vector<int32_t>* dly, int32_t* pos);

spiir_status compute_geometry(int T, int L, int S, int Dpad, int n, int opt_chunks, int nc_cap, int n_sm,
                              int smem_optin, FilterGeometry* g);
spiir_status kaiser_taps(int n_taps, double beta, double cutoff, float* out);

// worst quarter-warp conflict degree summed over all (group, slot, quarter), divided by their number
double layout_conflict_degree(const std::vector<int32_t>& dly, int G, int F);

}  // namespace spiir

// One class of templates that share a lane mapping (a uniform bank has exactly one).
struct spiir_bank_class {
    int T = 0, L = 0;                 // templates of the class, (largest) filters per template
    int F = 0, LPT = 0, TPG = 0, NP = 1, G = 0;
    size_t nfilt = 0;                 // G*F*32
    size_t state_off = 0;             // offset of the class inside a stream's state row (elements)
    int NC_cap = 1;                   // chunk scratch is sized for this many chunks
    float4* d_coef = nullptr;
    float2* d_apow = nullptr;         // a1^apow_C in d_coef's order: the in-CTA scan's chunk carry factor at n = max_block
    int apow_C = 0;
    int32_t* d_dly = nullptr;
    float2* d_chunk = nullptr;
    int32_t* d_tmap = nullptr;        // class template -> output row (nullptr for a uniform bank)
    double conflict_degree = 0.0;
};

struct spiir_plan {
    int T = 0, S = 1, rate_hz = 0, max_block = 0;
    int L_uniform = 0;                // > 0: uniform bank
    size_t n_filters_total = 0;       // sum over templates (caller order)
    int Dmax = 0, Dpad = 0;
    int opt_chunks = 0, flags = 0;
    spiir::DeviceInfo dev;
    std::vector<spiir_bank_class> cls;
    size_t nfilt_total = 0;           // sum of class nfilt: one stream's state row
    float2* d_state = nullptr;        // [S][nfilt_total]
    float* d_hist[2] = {nullptr, nullptr};   // [S][Dpad] ping-pong, shared by all classes
    int* d_phase = nullptr;           // {phase, arrivals}: which d_hist is current (flipped on the device)
    int32_t* d_pos = nullptr;         // [n_filters_total] caller filter -> index in the state row
    spiir::Arena arena;
};

struct spiir_resamp {
    int direction = 0, N = 0, rows = 0, max_block = 0;
    int H = 0;                        // history samples per row
    float* d_taps = nullptr;
    int flags = 0;                    // spiir_resamp_opts.flags
    void* d_hist[2] = {nullptr, nullptr};
    int* d_phase = nullptr;           // {phase, arrivals}
    std::vector<float> taps;
    spiir::DeviceInfo dev;
    spiir::Arena arena;
};

namespace spiir {
size_t plan_layout(spiir_plan* p, Arena* a);        // carves the plan's device buffers out of `a` (measuring arena: only sizes)
size_t resamp_layout(spiir_resamp* r, Arena* a);
spiir_status plan_geometry(const spiir_plan* p, const spiir_bank_class& c, int n, FilterGeometry* g);
spiir_status filter_launch(spiir_plan* p, const float* x, int n, spiir_c64* z, int accumulate, cudaStream_t st);
spiir_status filter_launch_group(spiir_plan* const* ps, const float* const* xs, const int* ns, spiir_c64* const* zs, int count,
                                 cudaStream_t st);
int plan_launches(const spiir_plan* p, int n);
spiir_status resamp_create_in(spiir_resamp_t** out, int direction, int n_taps, double kaiser_beta, double cutoff, int n_rows,
                              int max_block, Arena* parent, int flags = 0);
spiir_status plan_create_in(spiir_plan_t** out, const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays,
                            const int32_t* offsets, int n_templates, int n_filters, int rate_hz, const spiir_plan_opts& o,
                            Arena* parent);
spiir_status down_chain_launch(spiir_resamp* const* downs, int nstages, const float* x, int n, float* const* xh,
                               int n_streams, cudaStream_t st);
bool down_chain_fits(spiir_resamp* const* downs, int nstages, int n);
bool up_chain_fits(spiir_resamp* const* ups, int nstages, int n_low);
spiir_status up_chain_launch(spiir_resamp* const* ups, int nstages, const spiir_c64* z_low, int n_low,
                             const spiir_c64* const* z_add, spiir_c64* out, int rows, cudaStream_t st);
// resume state of a plan / stage as raw device copies (used by the multirate blob)
spiir_status plan_state_copy(spiir_plan* p, spiir_c64* y, float* hist, int to_user, cudaStream_t st);
spiir_status resamp_state_copy(spiir_resamp* r, void* hist, int to_user, cudaStream_t st);
}  // namespace spiir
