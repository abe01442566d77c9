// spiir_resamp.cu -- C ABI of libspiir.so, part 2: the x2 resampling stages (Eq. 9) and the
// fused down / up chains the multirate plan uses.  See include/spiir.h.
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <vector>

#include "spiir_internal.h"
#include "spiir_resample.cuh"
#include "spiir_resample_tc.cuh"

namespace spiir {

static size_t hist_bytes(const spiir_resamp* r)
{
    return (size_t)r->rows * std::max(1, r->H) * (r->direction == SPIIR_DOWN2 ? sizeof(float) : sizeof(float2));
}

size_t resamp_layout(spiir_resamp* r, Arena* a)
{
    const size_t start = a->used;
    r->d_phase = a->take_n<int>(64);
    r->d_taps = a->take_n<float>((size_t)r->N);
    r->d_hist[0] = a->take(hist_bytes(r));
    r->d_hist[1] = a->take(hist_bytes(r));
    a->used = (a->used + 255) & ~(size_t)255;
    return a->used - start;
}

static bool resamp_args_ok(int direction, int n_taps, int n_rows)
{
    return (direction == SPIIR_DOWN2 || direction == SPIIR_UP2) && n_taps >= 2 && n_taps <= kMaxTaps && !(n_taps & 1) && n_rows >= 1;
}

static void resamp_shape(spiir_resamp* r, int direction, int n_taps, int n_rows, int max_block)
{
    r->direction = direction; r->N = n_taps; r->rows = n_rows; r->max_block = max_block;
    r->H = direction == SPIIR_DOWN2 ? n_taps - 1 : n_taps / 2 - 1;
}

spiir_status resamp_create_in(spiir_resamp_t** out, int direction, int n_taps, double kaiser_beta, double cutoff, int n_rows,
                              int max_block, Arena* parent, int flags)
{
    *out = nullptr;
    spiir_resamp* r = new (std::nothrow) spiir_resamp;
    if (!r) return SPIIR_ENOMEM;
    r->taps.resize(n_taps);
    spiir_status rc = kaiser_taps(n_taps, kaiser_beta, cutoff, r->taps.data());
    if (rc == SPIIR_OK) rc = device_info(&r->dev);
    if (rc != SPIIR_OK) { delete r; return rc; }
    resamp_shape(r, direction, n_taps, n_rows, max_block);
    r->flags = flags;
    Arena probe;
    const size_t need = resamp_layout(r, &probe);
    r->arena.base = parent->base ? static_cast<char*>(parent->take(need)) : nullptr;
    r->arena.cap = need; r->arena.owned = false; r->arena.used = 0;
    if (!r->arena.base) { delete r; set_error("spiir_resamp_create: arena has no memory"); return SPIIR_ENOMEM; }
    resamp_layout(r, &r->arena);
    cudaError_t e = cudaMemset(r->d_phase, 0, 64 * sizeof(int));
    if (e == cudaSuccess) e = cudaMemcpy(r->d_taps, r->taps.data(), n_taps * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemset(r->d_hist[0], 0, hist_bytes(r));
    if (e == cudaSuccess) e = cudaMemset(r->d_hist[1], 0, hist_bytes(r));
    if (e != cudaSuccess) { rc = cuda_fail(e, "spiir_resamp_create initialisation"); delete r; return rc; }
    *out = r;
    return SPIIR_OK;
}

// history of a stage <-> the caller's [rows][H] buffer (current ping-pong half, resolved on the device)
template <typename T>
__global__ void spiir_resamp_hist_copy_kernel(T* h0, T* h1, const int* __restrict__ phase, T* user, size_t count, int to_user)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    T* cur = phase_read(phase) ? h1 : h0;
    if (to_user) user[i] = cur[i]; else cur[i] = user[i];
}

spiir_status resamp_state_copy(spiir_resamp* r, void* hist, int to_user, cudaStream_t st)
{
    if (r->H <= 0) return SPIIR_OK;
    const size_t count = (size_t)r->rows * r->H;
    const unsigned blocks = (unsigned)((count + 255) / 256);
    if (r->direction == SPIIR_DOWN2)
        spiir_resamp_hist_copy_kernel<float><<<blocks, 256, 0, st>>>(static_cast<float*>(r->d_hist[0]), static_cast<float*>(r->d_hist[1]),
                                                                      r->d_phase, static_cast<float*>(hist), count, to_user);
    else
        spiir_resamp_hist_copy_kernel<float2><<<blocks, 256, 0, st>>>(static_cast<float2*>(r->d_hist[0]), static_cast<float2*>(r->d_hist[1]),
                                                                       r->d_phase, static_cast<float2*>(hist), count, to_user);
    SPIIR_CUDA(cudaGetLastError());
    return SPIIR_OK;
}

template <int N, int R>
static spiir_status launch_down_fir(spiir_resamp* r, DownArgs d, int n_out, cudaStream_t st)
{
    DownTaps<N> t;
    memcpy(t.h, r->taps.data(), sizeof t.h);
    const int seg_max = 128 * R * (R < kDownR ? 2 : 1);  // outputs per row segment: one unit of R outputs per thread (two for small R)
    d.nseg = (n_out + seg_max - 1) / seg_max;
    d.seg = ((n_out + d.nseg - 1) / d.nseg + R - 1) / R * R;
    d.nseg = (n_out + d.seg - 1) / d.seg;
    const int w_len = (2 * d.seg + N - 1 + 2 * R + 7) & ~3;
    const size_t smem = (size_t)(w_len + d.seg) * sizeof(float);
    const dim3 grid(d.nseg * r->rows);
    SPIIR_CUDA(ensure_smem((const void*)spiir_down2_fir_kernel<N, R>, (int)smem));
    spiir_down2_fir_kernel<N, R><<<grid, 128, smem, st>>>(d, t);
    SPIIR_CUDA(cudaGetLastError());
    return SPIIR_OK;
}

// Tensor map of one call's input [rows][n_in] complex64, seen as rows of 2 n_in floats; box = 32 floats (16 samples) x
// ROWS rows with the 128-byte swizzle, zero fill outside the tensor.  cuTensorMapEncodeTiled is a host-side encoder (no
// driver call on the stream); it is resolved through the runtime so that the library does not link against libcuda.
static spiir_status up_tc_tensor_map(CUtensorMap* map, const void* in, int rows, int n_in)
{
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        SPIIR_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
        if (!fn || q != cudaDriverEntryPointSuccess) { set_error("cuTensorMapEncodeTiled is not available"); return SPIIR_ECUDA; }
        encode = reinterpret_cast<encode_fn>(fn);
    }
    const cuuint64_t dims[2] = {(cuuint64_t)2 * n_in, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)n_in * 8};
    const cuuint32_t box[2] = {32, (cuuint32_t)tc::ROWS};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult rc = encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(in), dims, strides, box, estr,
                               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (rc != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled failed (%d)", (int)rc); return SPIIR_ECUDA; }
    return SPIIR_OK;
}

template <int HALF>
static void fill_up_taps(const spiir_resamp* r, UpTaps<HALF>* t)
{
    for (int q = 0; q < HALF; ++q) { t->t0[q] = r->taps[2 * q]; t->t1[q] = r->taps[2 * q + 1]; }
}

}  // namespace spiir

using namespace spiir;

extern "C" {

void spiir_resamp_destroy(spiir_resamp_t* r)
{
    if (!r) return;
    arena_close(&r->arena);
    delete r;
}

size_t spiir_resamp_workspace_bytes(int direction, int n_taps, int n_rows)
{
    if (!resamp_args_ok(direction, n_taps, n_rows)) { set_error("spiir_resamp_workspace_bytes: bad arguments"); return 0; }
    spiir_resamp r;
    resamp_shape(&r, direction, n_taps, n_rows, 1);
    Arena probe;
    return resamp_layout(&r, &probe);
}

spiir_status spiir_resamp_create(spiir_resamp_t** out, int direction, int n_taps, double kaiser_beta, double cutoff,
                                 int n_rows, const spiir_resamp_opts* opts)
{
    if (!out) { set_error("spiir_resamp_create: out is NULL"); return SPIIR_EINVAL; }
    *out = nullptr;
    spiir_resamp_opts o = {4096, nullptr, 0, 0};
    if (opts) o = *opts;
    if (!resamp_args_ok(direction, n_taps, n_rows) || o.max_block < 1) {
        set_error("spiir_resamp_create: bad arguments");
        return SPIIR_EINVAL;
    }
    const size_t need = spiir_resamp_workspace_bytes(direction, n_taps, n_rows);
    Arena top;
    spiir_status rc = arena_open(&top, o.workspace, o.workspace_bytes, need, "spiir_resamp_create");
    if (rc != SPIIR_OK) return rc;
    rc = resamp_create_in(out, direction, n_taps, kaiser_beta, cutoff, n_rows, o.max_block, &top, o.flags);
    if (rc != SPIIR_OK) { arena_close(&top); return rc; }
    (*out)->arena.owned = top.owned;                      // the stage owns the block the library allocated for it
    return SPIIR_OK;
}

spiir_status spiir_resamp_reset(spiir_resamp_t* r, void* cuda_stream)
{
    if (!r) { set_error("spiir_resamp_reset: NULL"); return SPIIR_EINVAL; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    SPIIR_CUDA(cudaMemsetAsync(r->d_hist[0], 0, hist_bytes(r), st));
    SPIIR_CUDA(cudaMemsetAsync(r->d_hist[1], 0, hist_bytes(r), st));
    SPIIR_CUDA(cudaMemsetAsync(r->d_phase, 0, 2 * sizeof(int), st));
    return SPIIR_OK;
}

int spiir_resamp_history_len(const spiir_resamp_t* r) { return r ? r->H : 0; }

spiir_status spiir_resamp_get_state(spiir_resamp_t* r, void* hist_out, void* cuda_stream)
{
    if (!r || (!hist_out && r->H > 0)) { set_error("spiir_resamp_get_state: NULL argument"); return SPIIR_EINVAL; }
    return resamp_state_copy(r, hist_out, 1, static_cast<cudaStream_t>(cuda_stream));
}

spiir_status spiir_resamp_set_state(spiir_resamp_t* r, const void* hist_in, void* cuda_stream)
{
    if (!r || (!hist_in && r->H > 0)) { set_error("spiir_resamp_set_state: NULL argument"); return SPIIR_EINVAL; }
    return resamp_state_copy(r, const_cast<void*>(hist_in), 0, static_cast<cudaStream_t>(cuda_stream));
}

spiir_status spiir_resample_down(spiir_resamp_t* r, const float* in, int n_in, float* out, void* cuda_stream)
{
    if (!r || r->direction != SPIIR_DOWN2 || n_in < 0 || (n_in & 1)) { set_error("spiir_resample_down: bad plan or odd n_in"); return SPIIR_EINVAL; }
    if (n_in == 0) return SPIIR_OK;
    if (!in || !out) { set_error("spiir_resample_down: NULL buffer"); return SPIIR_EINVAL; }
    if (n_in > r->max_block) { set_error("spiir_resample_down: n_in exceeds max_block"); return SPIIR_ESTATE; }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (r->N == 384 || r->N == 192 || r->N == 32) {
        // register-blocked kernel, taps in the kernel parameters (constant bank)
        DownArgs d;
        d.in = in; d.out = out;
        d.hbuf[0] = reinterpret_cast<float*>(r->d_hist[0]); d.hbuf[1] = reinterpret_cast<float*>(r->d_hist[1]);
        d.phase = r->d_phase;
        d.rows = r->rows; d.n_in = n_in;
        const int n_out = n_in / 2;
        // outputs per thread: 6 for the long filters (lane stride 3 x 16 bytes: conflict-free; the unrolled body stays
        // inside the instruction cache: 384 taps at 10 outputs ran 5.6x slower), 10 for 32 taps
        if (r->N == 384) return launch_down_fir<384, 6>(r, d, n_out, st);
        if (r->N == 192) return launch_down_fir<192, 6>(r, d, n_out, st);
        return launch_down_fir<32, kDownR>(r, d, n_out, st);
    }
    ResampArgs a;
    a.taps = r->d_taps; a.in = in; a.out = out; a.hbuf[0] = r->d_hist[0]; a.hbuf[1] = r->d_hist[1]; a.phase = r->d_phase;
    a.rows = r->rows; a.n_in = n_in; a.N = r->N; a.accumulate = 0;
    const int n_out = n_in / 2;
    a.tile = std::min(512, (n_out + 127) / 128 * 128);
    const dim3 grid(r->rows, (n_out + a.tile - 1) / a.tile);
    const size_t smem = (size_t)(r->N + 2 * (a.tile + r->N / 2)) * sizeof(float);
    spiir_down2_kernel<<<grid, 128, smem, st>>>(a);
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
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    UpArgs u;
    u.in = reinterpret_cast<const float2*>(in); u.out = reinterpret_cast<float2*>(out);
    u.hbuf[0] = reinterpret_cast<float2*>(r->d_hist[0]); u.hbuf[1] = reinterpret_cast<float2*>(r->d_hist[1]);
    u.phase = r->d_phase;
    u.rows = r->rows; u.n_in = n_in; u.accumulate = accumulate;
    // 192 and 32 taps on the tensor cores (tcgen05: TF32 product + two bf16 correction products): FP32-bound (192) or
    // L1-bound (32) on the CUDA cores, HBM-bound here.  Needs enough work to fill the persistent CTAs; small calls keep
    // the CUDA-core kernels.
    if ((r->N == 192 || r->N == 32) && !(r->flags & 1) && (long long)r->rows * n_in >= 64LL * 1024) {
        tc::UpTcArgs t;
        t.in = u.in; t.out = u.out; t.hbuf[0] = u.hbuf[0]; t.hbuf[1] = u.hbuf[1]; t.phase = u.phase; t.taps = r->d_taps;
        t.rows = r->rows; t.n_in = n_in; t.accumulate = accumulate;
        t.tiles_per_row = (n_in + tc::TIN - 1) / tc::TIN;
        t.nstrips = (r->rows + tc::ROWS - 1) / tc::ROWS;
        // Time segments per strip: a unit (strip, segment) costs its tiles plus 1.5 tile-times of halo, the persistent CTAs
        // take the units round-robin; the segment length with the fewest tile-times on the busiest CTA wins (the shortest
        // on a tie: measured faster, 248 against 261 us on 16384 x 2048).
        {
            double best = 1e30;
            t.seg_tiles = t.tiles_per_row; t.nsegs = 1;
            for (int st_ = 1; st_ <= t.tiles_per_row; ++st_) {
                const int ns = (t.tiles_per_row + st_ - 1) / st_;
                const long units = (long)t.nstrips * ns;
                const long rounds = (units + r->dev.n_sm - 1) / r->dev.n_sm;
                const double cost = (double)rounds * (st_ + 1.5);
                if (cost < best * 0.999) { best = cost; t.seg_tiles = st_; t.nsegs = ns; }
            }
        }
        t.in16 = ((reinterpret_cast<uintptr_t>(in) & 15u) == 0 && (n_in & 1) == 0) ? 1 : 0;
        CUtensorMap in_map;
        memset(&in_map, 0, sizeof in_map);
        if (t.in16) {
            spiir_status mrc = up_tc_tensor_map(&in_map, in, r->rows, n_in);
            if (mrc != SPIIR_OK) return mrc;
        }
        const int grid = std::min(t.nstrips * t.nsegs, r->dev.n_sm);
        if (r->N == 192) {
            SPIIR_CUDA(ensure_smem((const void*)tc::spiir_up2_tc_kernel<96, 96>, tc::Geo<96, 96>::SMEM_BYTES));
            tc::spiir_up2_tc_kernel<96, 96><<<grid, tc::THREADS, tc::Geo<96, 96>::SMEM_BYTES, st>>>(t, in_map);
        } else {
            SPIIR_CUDA(ensure_smem((const void*)tc::spiir_up2_tc_kernel<32, 16>, tc::Geo<32, 16>::SMEM_BYTES));
            tc::spiir_up2_tc_kernel<32, 16><<<grid, tc::THREADS, tc::Geo<32, 16>::SMEM_BYTES, st>>>(t, in_map);
        }
        SPIIR_CUDA(cudaGetLastError());
        return SPIIR_OK;
    }
    // short filter: HBM-bound streaming kernel, no shared memory.  Its 16-byte input loads need 16-byte aligned rows
    // (in aligned and n_in even); other inputs take the register-blocked kernel below, which loads 8 bytes at a time.
    if (r->N == 32 && (reinterpret_cast<uintptr_t>(in) & 15u) == 0 && (n_in & 1) == 0) {
        u.seg = u.nseg = u.upr = u.rpc = 0;
        const long long units = (long long)r->rows * ((n_in + kUpSR - 1) / kUpSR);
        UpTaps<16> t;
        fill_up_taps<16>(r, &t);
        spiir_up2_stream_kernel<16><<<(unsigned)((units + 255) / 256), 256, 0, st>>>(u, t);
        SPIIR_CUDA(cudaGetLastError());
        return SPIIR_OK;
    }
    if (r->N == 192 || r->N == 32) {
        // register-blocked kernel, taps in the kernel parameters (constant bank)
        u.nseg = (n_in + kUpSegMax - 1) / kUpSegMax;
        u.seg = ((n_in + u.nseg - 1) / u.nseg + kUpR - 1) / kUpR * kUpR;
        u.nseg = (n_in + u.seg - 1) / u.seg;
        u.upr = u.seg / kUpR;
        const int half = r->N / 2;
        const int in_stride = (u.seg + half - 1 + kUpR + 3) & ~1, out_stride = 2 * (u.seg + kUpR);
        // rows per CTA: as many as 128 threads serve, but never more shared memory than the opt-in limit allows
        u.rpc = std::max(1, std::min(128 / u.upr, r->rows));
        while (u.rpc > 1 && (size_t)u.rpc * (in_stride + out_stride) * sizeof(float2) > (size_t)96 * 1024) --u.rpc;
        const size_t smem = (size_t)u.rpc * (in_stride + out_stride) * sizeof(float2);
        const dim3 grid(u.nseg * ((r->rows + u.rpc - 1) / u.rpc));
        if (half == 96) {
            UpTaps<96> t;
            fill_up_taps<96>(r, &t);
            SPIIR_CUDA(ensure_smem((const void*)spiir_up2_fir_kernel<96>, (int)smem));
            spiir_up2_fir_kernel<96><<<grid, 128, smem, st>>>(u, t);
        } else {
            UpTaps<16> t;
            fill_up_taps<16>(r, &t);
            SPIIR_CUDA(ensure_smem((const void*)spiir_up2_fir_kernel<16>, (int)smem));
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
    spiir_up2_kernel<<<grid, 128, smem, st>>>(a);
    SPIIR_CUDA(cudaGetLastError());
    return SPIIR_OK;
}

}  // extern "C"

namespace spiir {

// Row a8 in one launch: every down stage of a multirate plan (192 or 384 taps; the caller falls back to
// one spiir_resample_down per stage when this returns SPIIR_EUNSUPPORTED).
template <int N>
static spiir_status down_chain_launch_n(spiir_resamp* const* downs, const DownChainArgs& a, size_t smem, int n_streams, cudaStream_t st)
{
    DownTaps<N> t;
    memcpy(t.h, downs[0]->taps.data(), sizeof t.h);
    SPIIR_CUDA(ensure_smem((const void*)spiir_down_chain_kernel<N>, (int)smem));
    spiir_down_chain_kernel<N><<<n_streams, 512, smem, st>>>(a, t);
    SPIIR_CUDA(cudaGetLastError());
    return SPIIR_OK;
}

static bool down_chain_smem(spiir_resamp* const* downs, int nstages, int n, size_t* smem)
{
    const int N = downs[0]->N;
    if (nstages < 1 || nstages > kMaxStages || (N != 192 && N != 384)) return false;
    size_t words = 0;
    for (int k = 0; k <= nstages; ++k) words += down_chain_buf_len(N, n >> k);
    *smem = words * sizeof(float);
    return *smem <= (size_t)downs[0]->dev.smem_optin;
}

spiir_status down_chain_launch(spiir_resamp* const* downs, int nstages, const float* x, int n, float* const* xh,
                               int n_streams, cudaStream_t st)
{
    size_t smem = 0;
    if (!down_chain_smem(downs, nstages, n, &smem)) return SPIIR_EUNSUPPORTED;
    const int N = downs[0]->N;
    DownChainArgs a;
    a.x = x; a.n = n; a.nstages = nstages;
    for (int k = 0; k < nstages; ++k) {
        if (downs[k]->N != N || downs[k]->rows != n_streams) return SPIIR_EUNSUPPORTED;
        a.xh[k] = xh[k];
        a.hbuf[k][0] = reinterpret_cast<float*>(downs[k]->d_hist[0]);
        a.hbuf[k][1] = reinterpret_cast<float*>(downs[k]->d_hist[1]);
        a.phase[k] = downs[k]->d_phase;
    }
    return N == 192 ? down_chain_launch_n<192>(downs, a, smem, n_streams, st) : down_chain_launch_n<384>(downs, a, smem, n_streams, st);
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
        fill_up_taps<96>(ups[0], &t);
        SPIIR_CUDA(ensure_smem((const void*)spiir_up_chain_kernel<96>, (int)smem));
        spiir_up_chain_kernel<96><<<rows, 128, smem, st>>>(a, t);
    } else {
        UpTaps<16> t;
        fill_up_taps<16>(ups[0], &t);
        SPIIR_CUDA(ensure_smem((const void*)spiir_up_chain_kernel<16>, (int)smem));
        spiir_up_chain_kernel<16><<<rows, 128, smem, st>>>(a, t);
    }
    SPIIR_CUDA(cudaGetLastError());
    return SPIIR_OK;
}

// Whether the fused chains can serve a block of n base-rate samples (same conditions as the launchers).
bool down_chain_fits(spiir_resamp* const* downs, int nstages, int n)
{
    size_t smem = 0;
    return down_chain_smem(downs, nstages, n, &smem);
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
