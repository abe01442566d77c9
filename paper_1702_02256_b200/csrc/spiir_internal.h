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

// Launch geometry of the filter kernel for one block length (host logic, testable without a GPU).
struct FilterGeometry {
    int F, LPT, TPG, G;       // filters per lane, lanes per template, templates per group, groups
    int NC, C;                // time chunks and chunk length
    int NT, CS;               // time tile and shifted-copy stride (floats)
    int warps, grid_x, grid_y;
    int smem_bytes;
    int launches;
};

// Pick (F, LPT) for a bank of L filters per template.  Returns false when L is not supported.
bool choose_lane_mapping(int L, int T, int* F, int* LPT);
int lpt16_min_templates();

// Position (index into the [G][F][32] plan arrays) of every filter [T][L]; fills the permuted
// coefficient / delay arrays (zero padded).  avoid_conflicts: spread the 16-byte bank groups of
// the window reads over each quarter warp.
void build_layout(const spiir_c64* a1, const spiir_c64* b0, const int32_t* delays, int T, int L, int F, int LPT,
                  bool avoid_conflicts, std::vector<float>* coef /* [G*F*32*4] */, std::vector<int32_t>* dly,
                  std::vector<int32_t>* pos /* [T*L] */);

spiir_status compute_geometry(int T, int L, int S, int Dpad, int n, int opt_chunks, int nc_cap, int n_sm,
                              int smem_optin, FilterGeometry* g);
spiir_status kaiser_taps(int n_taps, double beta, double cutoff, float* out);

// worst quarter-warp conflict degree summed over all (group, slot, quarter), divided by their number
double layout_conflict_degree(const std::vector<int32_t>& dly, int G, int F);

}  // namespace spiir

struct spiir_plan {
    int T = 0, L = 0, S = 1, rate_hz = 0, max_block = 0;
    int Dmax = 0, Dpad = 0;
    int F = 0, LPT = 0, TPG = 0, G = 0;
    size_t nfilt = 0;                 // G*F*32
    int opt_chunks = 0, flags = 0;
    int NC_cap = 1;                   // chunk scratch is sized for this many chunks
    spiir::DeviceInfo dev;
    float4* d_coef = nullptr;
    int32_t* d_dly = nullptr;
    float2* d_state = nullptr;
    float2* d_chunk = nullptr;
    float* d_hist[2] = {nullptr, nullptr};
    int* d_phase = nullptr;           // {phase, arrivals}: which d_hist is current (flipped on the device)
    int32_t* d_pos = nullptr;
    double conflict_degree = 0.0;
};

struct spiir_resamp {
    int direction = 0, N = 0, rows = 0, max_block = 0;
    int H = 0;                        // history samples per row
    float* d_taps = nullptr;
    void* d_hist[2] = {nullptr, nullptr};
    int* d_phase = nullptr;           // {phase, arrivals}
    std::vector<float> taps;
    spiir::DeviceInfo dev;
};

namespace spiir {
spiir_status plan_geometry(const spiir_plan* p, int n, FilterGeometry* g);
spiir_status filter_launch(spiir_plan* p, const float* x, int n, spiir_c64* z, int accumulate, cudaStream_t st);
spiir_status filter_launch_group(spiir_plan* const* ps, const float* const* xs, const int* ns, spiir_c64* const* zs, int count,
                                 cudaStream_t st);
spiir_status down_chain_launch(spiir_resamp* const* downs, int nstages, const float* x, int n, float* const* xh,
                               int n_streams, cudaStream_t st);
bool down_chain_fits(spiir_resamp* const* downs, int nstages, int n);
bool up_chain_fits(spiir_resamp* const* ups, int nstages, int n_low);
spiir_status up_chain_launch(spiir_resamp* const* ups, int nstages, const spiir_c64* z_low, int n_low,
                             const spiir_c64* const* z_add, spiir_c64* out, int rows, cudaStream_t st);
}  // namespace spiir
