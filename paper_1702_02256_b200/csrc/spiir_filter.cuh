// spiir_filter.cuh -- sm_100a kernels for the single-rate SPIIR bank (Eq. 7 + Eq. 8).
//
// Mapping:
//   * a warp task = one "group" of 32/LPT templates; LPT lanes share a template and every lane
//     owns F filters of it, so a template's L <= F*LPT filters live in registers (a1, b0, y).
//   * the strain window x[t0-Dpad .. t0+NT) of the CTA's stream is staged ONCE into shared
//     memory with TMA bulk copies (cp.async.bulk + mbarrier), then replicated into four copies
//     shifted by 0..3 samples so that every filter, whatever its delay, fetches four consecutive
//     time steps with one aligned 16-byte LDS (row a1/a2 of SURVEY.md section 8).
//   * Eq. 7 is evaluated with packed FP32 pairs (FFMA2/FMUL2/FADD2, sm_100a): the pair is
//     (re, im), x and the coefficients enter as broadcast operands -- 4 packed instructions per
//     filter-sample update instead of 8 scalar ones.
//   * Eq. 8: per lane the F filters are summed in registers; 16 time steps are batched and summed
//     across the lanes of the template with a transposed butterfly (xor-shuffles), which leaves every
//     lane with a distinct slice of the 16 complex outputs -> coalesced stores, fixed summation order.
//   * templates of more than 512 filters span NP adjacent warps of one CTA (the
//     513-filter example): every warp transposes its partial sums through a padded, conflict-free
//     shared-memory tile and the NP partial results meet there behind one named barrier per batch.
//   * time-parallel mode (row a7): a block is cut into chunks; pass 1 runs every chunk from zero
//     state (chunk 0 from the carried state), a carry kernel propagates s_{c+1} = a1^C s_c + e_c,
//     pass 2 reruns every chunk from its true initial state and writes z.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "spiir_common.cuh"

namespace spiir {

constexpr int kBatch = 16;        // time steps per reduction batch
constexpr int kMaxWarps = 8;      // warps per CTA (launch bound 256 threads -> up to 255 registers)

struct FilterArgs {
    const float4* coef;      // [G][F][32]  (a1.re, a1.im, b0.re, b0.im), plan order
    const int*    dly;       // [G][F][32]  delay in samples
    const float2* apow;      // [G][F][32]  a1^C for this launch's chunk length C (in-CTA scan), or nullptr: computed in the kernel
    float2*       state;     // [S][sstride], this bank's [G][F][32] carried y (in/out) at the start of every row
    size_t        sstride;   // elements between the state rows of two streams
    float2*       chunk_st;  // chunked modes: [S][NC][G][F][32]; pass 1 writes end states, carry
                             // turns them into initial states in place, pass 2 reads them
    float*        hbuf[2];   // [S][Dpad] input history, ping-pong: hbuf[phase] holds the Dpad samples before
                             // this block (oldest first), hbuf[phase ^ 1] is written in slices by the CTAs of stream s
    int*          phase;     // device words {phase, arrivals}: which buffer is current is decided on the
                             // device, so that every call enqueues identical work (CUDA-graph replayable)
    const float*  x;         // [S][n]
    float2*       z;         // [S][T][n]
    int n, T, G, S;
    int Dpad;                // history length, multiple of 4, >= max delay
    int NT;                  // time-tile length (multiple of kBatch) staged per window
    int CS;                  // stride between the shifted window copies, floats, multiple of 4
    int NC;                  // time chunks (1 = plain streaming)
    int C;                   // chunk length (multiple of kBatch); chunk c covers [c*C, min(n,(c+1)*C))
    int mode;                // 0 plain, 1 chunk pass 1 (no z), 2 chunk pass 2
    int x_aligned;           // x rows are 16-byte aligned (x pointer and n*4) -> TMA path
    int accumulate;          // z += result instead of z = result
    const int* tmap;         // ragged plans: output row of template t of this class (nullptr: row = t)
    int T_rows;              // rows of z per stream (= T unless the bank is one class of a ragged plan)
    int NP;                  // warps per template (LPT = 32 only; G = T * NP pieces)
    int carry;               // this launch writes the next input history and flips the phase
    int z16;                 // every row of z starts 16-byte aligned (z pointer and n even): few-filter mappings store full lines
};

// shared-memory scratch of one warp for the transposed reduction (LPT = 32), in float4 units:
// [32 rows][9] (a row = the lane's 16 complex partial sums + one float4 of padding) and [2][32] second-stage words
constexpr int kRedRows4 = 32 * 9;
constexpr int kRedWarp4 = kRedRows4 + 64;

__device__ __forceinline__ void named_bar_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// ---------------------------------------------------------------------------------------------
// PTX helpers: mbarrier + TMA bulk copy (global -> shared)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE;\n"
        "bra WAIT_LOOP;\n"
        "DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// ---------------------------------------------------------------------------------------------
// Window staging.  W[i], i in [0, Dpad+len_pad): sample g = t0 - Dpad + i of stream s
// (g < 0 -> history, 0 <= g < n -> x, else 0).  Copy s holds W shifted by s: copy_s[i] = W[i+s].
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void stage_window(float* win, uint64_t* bar, uint32_t& parity, const FilterArgs& a,
                                             const float* __restrict__ hist_s, const float* __restrict__ x_s,
                                             int t0)
{
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int CS = a.CS, Dpad = a.Dpad, n = a.n;
    // valid samples: i in [0, nv) where nv = Dpad + min(NT, n - t0)
    const int nA = (t0 < Dpad) ? (Dpad - t0) : 0;           // samples taken from the history
    const int gB = t0 - Dpad + nA;                            // first x sample (>= 0)
    int nB = min(a.NT, n - t0) + (Dpad - nA);                 // samples taken from x
    const int nv = nA + nB;
    const bool use_tma = a.x_aligned != 0;
    int nB_tma = 0;
    if (use_tma) {
        nB_tma = nB & ~3;
        if (tid == 0) {
            uint32_t bytes = (uint32_t)(nA + nB_tma) * 4u;
            if (bytes) {
                mbar_expect_tx(bar, bytes);
                if (nA) tma_bulk_g2s(win, hist_s + t0, (uint32_t)nA * 4u, bar);
                if (nB_tma) tma_bulk_g2s(win + nA, x_s + gB, (uint32_t)nB_tma * 4u, bar);
            }
        }
        for (int i = nA + nB_tma + tid; i < nv; i += nthr) win[i] = x_s[gB + (i - nA)];
    } else {
        for (int i = tid; i < nv; i += nthr) win[i] = (i < nA) ? hist_s[t0 + i] : x_s[gB + (i - nA)];
    }
    for (int i = nv + tid; i < CS; i += nthr) win[i] = 0.f;   // zero tail (ragged block / shift overrun)
    if (use_tma && (nA + nB_tma) > 0) { mbar_wait(bar, parity); parity ^= 1u; }
    __syncthreads();
    // shifted copies 1..3 from copy 0, 16-byte accesses only
    const float4* w4 = reinterpret_cast<const float4*>(win);
    const int n4 = CS >> 2;
    for (int j = tid; j < n4 - 1; j += nthr) {
        float4 v0 = w4[j], v1 = w4[j + 1];
        reinterpret_cast<float4*>(win + CS)[j]     = make_float4(v0.y, v0.z, v0.w, v1.x);
        reinterpret_cast<float4*>(win + 2 * CS)[j] = make_float4(v0.z, v0.w, v1.x, v1.y);
        reinterpret_cast<float4*>(win + 3 * CS)[j] = make_float4(v0.w, v1.x, v1.y, v1.z);
    }
    if (tid == 0) {
        const float4 zq = make_float4(0.f, 0.f, 0.f, 0.f);
        reinterpret_cast<float4*>(win + CS)[n4 - 1] = zq;
        reinterpret_cast<float4*>(win + 2 * CS)[n4 - 1] = zq;
        reinterpret_cast<float4*>(win + 3 * CS)[n4 - 1] = zq;
    }
    __syncthreads();
}

// ---------------------------------------------------------------------------------------------
// Transposed butterfly: Z[0..15] per lane (partial sums of 16 time steps) -> sums over the LPT
// lanes of a template; afterwards lane j of the template holds steps [j*16/LPT, (j+1)*16/LPT)
// (LPT = 32: lane j holds float j of the 32 floats).
// ---------------------------------------------------------------------------------------------
template <int N, int M>
__device__ __forceinline__ void bfly_stage(float2* Z, int lane)
{
    const bool up = (lane & M) != 0;
#pragma unroll
    for (int i = 0; i < N / 2; ++i) {
        float2 lo = Z[i], hi = Z[i + N / 2];
        float2 keep = up ? hi : lo;
        float2 send = up ? lo : hi;
        float2 r;
        r.x = __shfl_xor_sync(0xffffffffu, send.x, M);
        r.y = __shfl_xor_sync(0xffffffffu, send.y, M);
        Z[i] = __fadd2_rn(keep, r);
    }
}

struct RedCtx {
    float4* rows;            // this warp's [32][9] tile
    float4* part2;           // this warp's [2][32] second-stage words
    int part, NP, bar_id;    // piece index within the template, pieces per template, named barrier of the template
};

// LPT = 32.  Every lane writes its 16 complex partial sums as one padded row; lane j then sums float quad (j & 7)
// over the eight rows 4i + (j >> 3); the four partial quads of a column meet in a second tile, from which lane j
// sums float j.  With NP > 1 the second tiles of the NP warps of a template are summed by its first warp after a
// named barrier (double-buffered by the batch parity, so one barrier per batch suffices).
template <bool MULTI>
__device__ __forceinline__ void reduce_store_warp(float2 (&Z)[kBatch], int lane, float2* zrow, int nvalid, bool active, bool acc,
                                                  const RedCtx& rc, int bpar)
{
    // One warp per template: the xor-butterfly.  (A shared-memory transposition needs a third of the instructions but
    // measured 3 % slower in this kernel: the window reads already keep the shared-memory pipe ~55 % busy.)
    if (!MULTI) {
        bfly_stage<16, 16>(Z, lane); bfly_stage<8, 8>(Z, lane); bfly_stage<4, 4>(Z, lane); bfly_stage<2, 2>(Z, lane);
        const bool up = (lane & 1) != 0;
        float keep = up ? Z[0].y : Z[0].x;
        float send = up ? Z[0].x : Z[0].y;
        float v = keep + __shfl_xor_sync(0xffffffffu, send, 1);
        if (active && (lane >> 1) < nvalid) {
            float* p = reinterpret_cast<float*>(zrow) + lane;
            if (acc) v += *p;
            *p = v;
        }
        return;
    }
    float4* myrow = rc.rows + lane * 9;
#pragma unroll
    for (int q = 0; q < 8; ++q) myrow[q] = make_float4(Z[2 * q].x, Z[2 * q].y, Z[2 * q + 1].x, Z[2 * q + 1].y);
    __syncwarp();
    const float4* col = rc.rows + (lane >> 3) * 9 + (lane & 7);
    float2 a0 = make_float2(0.f, 0.f), a1 = make_float2(0.f, 0.f);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float4 v = col[i * 36];
        a0 = __fadd2_rn(a0, make_float2(v.x, v.y));
        a1 = __fadd2_rn(a1, make_float2(v.z, v.w));
    }
    rc.part2[bpar * 32 + lane] = make_float4(a0.x, a0.y, a1.x, a1.y);
    named_bar_sync(rc.bar_id, 32 * rc.NP);
    if (rc.part != 0) return;
    float v = 0.f;
    for (int p = 0; p < rc.NP; ++p) {
        const float* f = reinterpret_cast<const float*>(rc.part2 + (size_t)p * kRedWarp4 + bpar * 32);
        const float w = (f[lane] + f[32 + lane]) + (f[64 + lane] + f[96 + lane]);
        v = p == 0 ? w : v + w;
    }
    if (active && (lane >> 1) < nvalid) {
        float* o = reinterpret_cast<float*>(zrow) + lane;
        if (acc) v += *o;
        *o = v;
    }
}

template <int LPT>
__device__ __forceinline__ void reduce_store(float2 (&Z)[kBatch], int lane, float2* zrow, int nvalid, bool active, bool acc)
{
    static_assert(LPT < 32, "one warp per template reduces through shared memory (reduce_store_warp)");
    // zrow: this lane's template row at the batch start (complex index), valid when active
    if (LPT >= 2)  bfly_stage<16, LPT / 2>(Z, lane);
    if (LPT >= 4)  bfly_stage<8, LPT / 4>(Z, lane);
    if (LPT >= 8)  bfly_stage<4, LPT / 8>(Z, lane);
    if (LPT >= 16) bfly_stage<2, LPT / 16>(Z, lane);
    constexpr int NV = kBatch / LPT;                  // complex values left per lane
    const int base = (lane & (LPT - 1)) * NV;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        if (active && base + i < nvalid) {
            float2 v = Z[i];
            if (acc) { float2 o = zrow[base + i]; v.x += o.x; v.y += o.y; }
            zrow[base + i] = v;
        }
    }
}

// Few lanes per template (LPT <= 4): after the butterfly a lane holds 16/LPT consecutive outputs of ITS template, so a
// direct store makes every lane of a warp instruction hit a different 128-byte line with 8..32 bytes (row a5 is the bound
// of this regime: 512 sector writes per batch).  Instead the warp's [32/LPT templates][16 steps] tile goes
// through shared memory (rows padded to 144 bytes: conflict-free both ways) and is written as whole 128-byte lines,
// eight lanes per row.  trow[i]: output row of tile row 4i + lane/8, or -1.
constexpr int kTileRow4 = 9;                                   // float4 per tile row (8 + 1 padding)
template <int LPT>
__device__ __forceinline__ void reduce_store_tile(float2 (&Z)[kBatch], int lane, float4* tile, float2* z_s, size_t n, int tpos,
                                                  const int (&trow)[(32 / LPT + 3) / 4], int nvalid, bool acc)
{
    static_assert(LPT <= 4, "wider mappings already store contiguous 16-byte pieces");
    if (LPT >= 2) bfly_stage<16, LPT / 2>(Z, lane);
    if (LPT >= 4) bfly_stage<8, LPT / 4>(Z, lane);
    constexpr int NV = kBatch / LPT;                           // complex values per lane
    float4* my = tile + (lane / LPT) * kTileRow4 + (lane % LPT) * (NV / 2);
#pragma unroll
    for (int i = 0; i < NV / 2; ++i) my[i] = make_float4(Z[2 * i].x, Z[2 * i].y, Z[2 * i + 1].x, Z[2 * i + 1].y);
    __syncwarp();
    const int q = lane & 7;
#pragma unroll
    for (int i = 0; i < (32 / LPT + 3) / 4; ++i) {
        if (trow[i] >= 0 && 2 * q < nvalid) {
            float4 v = tile[(4 * i + (lane >> 3)) * kTileRow4 + q];
            float2* dst = z_s + (size_t)trow[i] * n + tpos + 2 * q;
            if (2 * q + 1 < nvalid) {
                if (acc) { const float4 o = *reinterpret_cast<const float4*>(dst); v.x += o.x; v.y += o.y; v.z += o.z; v.w += o.w; }
                *reinterpret_cast<float4*>(dst) = v;
            } else {
                if (acc) { v.x += dst->x; v.y += dst->y; }
                *dst = make_float2(v.x, v.y);
            }
        }
    }
    __syncwarp();
}

// Where a batch of 16 outputs goes: one entry point for the three reductions above.
template <int LPT>
struct OutCtx {
    static constexpr int NI = LPT <= 4 ? (32 / LPT + 3) / 4 : 1;
    float2* zt;          // this lane's template row at the block start (valid when active)
    float2* z_s;         // row 0 of this stream
    size_t n;
    float4* tile;        // LPT <= 4: this warp's [32/LPT][kTileRow4] tile
    int trow[NI];        // LPT <= 4: output row of tile row 4i + lane/8, or -1
    bool active, acc, z16;
};

template <int LPT>
__device__ __forceinline__ void out_ctx_rows(OutCtx<LPT>& o, const FilterArgs& a, int g, int lane)
{
    constexpr int TPG = 32 / LPT;
#pragma unroll
    for (int i = 0; i < OutCtx<LPT>::NI; ++i) {
        const int r = 4 * i + (lane >> 3), tl = g * TPG + r;
        o.trow[i] = (LPT <= 4 && r < TPG && tl < a.T) ? (a.tmap ? a.tmap[tl] : tl) : -1;
    }
}

template <int LPT, bool MULTI>
__device__ __forceinline__ void emit_batch(float2 (&Z)[kBatch], int lane, int tpos, int nvalid, const OutCtx<LPT>& o,
                                           const RedCtx& rc, int bpar)
{
    if constexpr (LPT == 32) {
        reduce_store_warp<MULTI>(Z, lane, o.zt + tpos, nvalid, o.active, o.acc, rc, bpar);
    } else if constexpr (LPT <= 4) {
        if (o.z16) reduce_store_tile<LPT>(Z, lane, o.tile, o.z_s, o.n, tpos, o.trow, nvalid, o.acc);
        else reduce_store<LPT>(Z, lane, o.zt + tpos, nvalid, o.active, o.acc);
    } else {
        reduce_store<LPT>(Z, lane, o.zt + tpos, nvalid, o.active, o.acc);
    }
}

// ---------------------------------------------------------------------------------------------
// 16 time steps of Eq. 7 for the F filters of a lane.  off4[f]: float4 index of W[Dpad + j - d_f]
// in the right shifted copy at batch start j.
// ---------------------------------------------------------------------------------------------
template <int F, bool FULL, bool NOZ>
__device__ __forceinline__ void batch_steps(const float4* __restrict__ win4, const int (&off4)[F], int j4,
                                            const float4 (&cf)[F], float2 (&Y)[F], float2 (&Z)[kBatch], int nvalid)
{
#pragma unroll
    for (int q = 0; q < kBatch / 4; ++q) {
        float4 xv[F];
#pragma unroll
        for (int f = 0; f < F; ++f) xv[f] = win4[off4[f] + j4 + q];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int step = 4 * q + u;
            if (FULL || step < nvalid) {
                // y' = a1*y + b0*x as (re, im) pair arithmetic; the three instructions of a filter are
                // dependent, so they are issued breadth-first over the F filters of the lane
                float2 t[F];
#pragma unroll
                for (int f = 0; f < F; ++f) {
                    const float xs = (u == 0) ? xv[f].x : (u == 1) ? xv[f].y : (u == 2) ? xv[f].z : xv[f].w;
                    t[f] = __fmul2_rn(make_float2(cf[f].z, cf[f].w), make_float2(xs, xs));
                }
#pragma unroll
                for (int f = 0; f < F; ++f) t[f] = __ffma2_rn(make_float2(cf[f].x, cf[f].x), Y[f], t[f]);
                // (-yi, yr) * (ai, ai): the half-negated swap rides on the operand modifiers of FFMA2
#pragma unroll
                for (int f = 0; f < F; ++f) Y[f] = __ffma2_rn(make_float2(-Y[f].y, Y[f].x), make_float2(cf[f].y, cf[f].y), t[f]);
                if (!NOZ) {
                    // Eq. 8 within the lane: pairwise tree over the F filters (fixed order)
#pragma unroll
                    for (int f = 0; f < F; ++f) t[f] = Y[f];
#pragma unroll
                    for (int w = 1; w < F; w *= 2)
#pragma unroll
                        for (int f = 0; f + w < F; f += 2 * w) t[f] = __fadd2_rn(t[f], t[f + w]);
                    Z[step] = t[0];
                }
            } else if (!NOZ) {
                Z[step] = make_float2(0.f, 0.f);
            }
        }
    }
}

// The kernel body takes its CTA coordinates as arguments so that one launch can also serve several banks
// (spiir_filter_multi_kernel below): bx in [0, gdx), by in [0, gdy) with gdy = S * NC.
template <int F, int LPT, bool NOZ, bool MULTI>
__device__ __forceinline__ void filter_body(const FilterArgs& a, const int bx, const int by, const int gdx, const int gdy)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* win = reinterpret_cast<float*>(smem_raw);                   // 4 copies x CS floats
    uint64_t* bar = reinterpret_cast<uint64_t*>(win + 4 * (size_t)a.CS);
    float4* red = reinterpret_cast<float4*>(win + 4 * (size_t)a.CS + 4);    // multi-warp templates: kRedWarp4 float4 per warp; LPT <= 4: store tiles

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int s = by / a.NC, c = by % a.NC;
    const int tc0 = c * a.C;                                            // chunk range [tc0, tc1)
    const int tc1 = min(a.n, tc0 + a.C);
    // ONE thread reads the phase word and then adds the CTA's share (same address, program order); everybody else takes
    // the value from shared memory.  A thread that read the word itself could do so after the launch's last share had
    // landed -- nothing orders the warps of a CTA between the read and the add -- and see the NEXT phase.
    // The value is handed over only in front of the first window (below): its DRAM round trip overlaps the first
    // group's coefficient / state loads.
    int* sph = reinterpret_cast<int*>(bar + 1);                          // the 8 bytes behind the mbarrier are free
    uint32_t parity = 0;
    int ph = 0;
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        ph = phase_parity(a.phase);
        if (a.carry) phase_arrive(a.phase, by * gdx + bx, gdx * gdy);    // no one waits for this
    }
    __syncthreads();
    bool ph_known = false;
    const float* hist_s = nullptr;
    const float* x_s = a.x + (size_t)s * a.n;
    const int ntiles = (tc1 - tc0 + a.NT - 1) / a.NT;
    // single-tile case: the window is staged once, AFTER the first group's coefficient / state loads have been
    // issued (below), so that their DRAM round trip overlaps the TMA copy and the shifted copies
    bool staged = ntiles != 1;
    const float4* win4 = reinterpret_cast<const float4*>(win);

    constexpr int TPG = 32 / LPT;                                       // templates per group
    const int NP = MULTI ? a.NP : 1;                                    // warps per template (nwarps % NP == 0)
    RedCtx rc;
    rc.NP = NP; rc.part = warp % NP; rc.bar_id = 1 + warp / NP;
    rc.rows = red + (size_t)warp * kRedWarp4;
    rc.part2 = rc.rows + kRedRows4;      // the pieces of a template are adjacent warps: piece p's words sit p * kRedWarp4 on
    int bcount = 0;                                                     // batches done (parity = second-stage buffer)
    for (int g0 = bx * nwarps; g0 < a.G; g0 += gdx * nwarps) {
        const int g = g0 + warp;                                        // piece: template g / NP, part g % NP
        const bool wactive = g < a.G;
        const int tl = (g / NP) * TPG + lane / LPT;                     // template within this bank
        const bool active = wactive && tl < a.T;
        const int t = active ? (a.tmap ? a.tmap[tl] : tl) : 0;          // output row
        float4 cf[F]; float2 Y[F]; int off4[F];
        const size_t lbase = ((size_t)(wactive ? g : 0) * F) * 32 + lane;
        // All 3 F loads of the lane are issued before any of them is used, from ONE address per array chosen without a
        // branch.  (With the delay consumed inside the loop and the state behind an if / else, ptxas kept the loop order:
        // F DRAM round trips in a row, 6 us of the 9.5 us prologue of configs[1].)
        const float2* ysrc = a.mode == 2 ? a.chunk_st + (((size_t)s * a.NC + c) * a.G * F) * 32 + lbase
                                         : a.state + (size_t)s * a.sstride + lbase;
        const bool yload = wactive && (a.mode == 0 || a.mode == 2 || (a.mode == 1 && c == 0));
        int dl[F];
#pragma unroll
        for (int f = 0; f < F; ++f) {
            cf[f] = wactive ? a.coef[lbase + (size_t)f * 32] : make_float4(0.f, 0.f, 0.f, 0.f);
            dl[f] = wactive ? a.dly[lbase + (size_t)f * 32] : 0;
            Y[f] = yload ? ysrc[(size_t)f * 32] : make_float2(0.f, 0.f);
        }
        OutCtx<LPT> oc;
        oc.zt = active ? a.z + ((size_t)s * a.T_rows + t) * (size_t)a.n : nullptr;
        oc.z_s = a.z + (size_t)s * a.T_rows * (size_t)a.n; oc.n = (size_t)a.n;
        oc.tile = red + (size_t)warp * (TPG * kTileRow4);
        oc.active = active; oc.acc = a.accumulate != 0; oc.z16 = a.z16 != 0;
        out_ctx_rows<LPT>(oc, a, g, lane);
        if (!ph_known) {                                                // first group only (uniform over the CTA)
            if (threadIdx.x == 0) *sph = ph;
            __syncthreads();
            ph = *sph;
            hist_s = a.hbuf[ph] + (size_t)s * a.Dpad;
            ph_known = true;
        }
        if (!staged) { stage_window(win, bar, parity, a, hist_s, x_s, tc0); staged = true; }
        // first use of the loads above: they were in flight while the window was staged
#pragma unroll
        for (int f = 0; f < F; ++f) {
            const int sh = (-dl[f]) & 3;
            off4[f] = (sh * a.CS + a.Dpad - dl[f] - sh) >> 2;
        }

        for (int tile = 0; tile < ntiles; ++tile) {
            const int t0 = tc0 + tile * a.NT;
            const int len = min(a.NT, tc1 - t0);
            if (ntiles > 1) { __syncthreads(); stage_window(win, bar, parity, a, hist_s, x_s, t0); }
            const int nfull = len / kBatch;
            float2 Z[kBatch];
            for (int b = 0; b < nfull; ++b) {
                batch_steps<F, true, NOZ>(win4, off4, b * (kBatch / 4), cf, Y, Z, kBatch);
                if (!NOZ) { emit_batch<LPT, MULTI>(Z, lane, t0 + b * kBatch, kBatch, oc, rc, bcount & 1); ++bcount; }
            }
            const int rem = len - nfull * kBatch;
            if (rem > 0) {
                batch_steps<F, false, NOZ>(win4, off4, nfull * (kBatch / 4), cf, Y, Z, rem);
                if (!NOZ) { emit_batch<LPT, MULTI>(Z, lane, t0 + nfull * kBatch, rem, oc, rc, bcount & 1); ++bcount; }
            }
        }
        if (wactive) {
#pragma unroll
            for (int f = 0; f < F; ++f) {
                if (a.mode == 0 || (a.mode == 2 && c == a.NC - 1))
                    a.state[(size_t)s * a.sstride + lbase + (size_t)f * 32] = Y[f];
                else if (a.mode == 1)
                    a.chunk_st[(((size_t)s * a.NC + c) * a.G * F) * 32 + lbase + (size_t)f * 32] = Y[f];
            }
        }
    }
    // carried history for the next block (reads only hist + x, writes the other buffer: no race with other CTAs).  Every
    // CTA of the stream copies a slice, at the END of its life: by then x and the history are in L2 and the copy is off
    // the critical path (at the top it was a chain of DRAM round trips in front of the coefficient loads).
    if (!ph_known) {                                                    // a CTA without a group (cannot happen with the host's grids)
        if (threadIdx.x == 0) *sph = ph;
        __syncthreads();
        ph = *sph;
        hist_s = a.hbuf[ph] + (size_t)s * a.Dpad;
    }
    if (a.carry) {
        float* hn = a.hbuf[ph ^ 1] + (size_t)s * a.Dpad;
        const int cta = c * gdx + bx, nctas = a.NC * gdx;
        if (a.NC == 1 && ntiles == 1 && staged) {      // the window still holds the whole block: W[n + i] is sample n - Dpad + i
            for (int i = cta * blockDim.x + threadIdx.x; i < a.Dpad; i += nctas * blockDim.x) hn[i] = win[a.n + i];
        } else {
            for (int i = cta * blockDim.x + threadIdx.x; i < a.Dpad; i += nctas * blockDim.x) {
                int g = a.n - a.Dpad + i;
                hn[i] = (g >= 0) ? x_s[g] : hist_s[a.n + i];
            }
        }
    }
}

template <int F, int LPT, bool NOZ, bool MULTI = false>
__global__ void __launch_bounds__(kMaxWarps * 32) spiir_filter_kernel(const FilterArgs a)
{
    static_assert(!MULTI || LPT == 32, "only whole-warp templates span several warps");
    filter_body<F, LPT, NOZ, MULTI>(a, blockIdx.x, blockIdx.y, gridDim.x, gridDim.y);
}

// ---------------------------------------------------------------------------------------------
// Time-parallel scan INSIDE one CTA (row a7 for banks that cannot fill the machine and whose blocks are
// too short to pay for three launches: the few-filter regime, and the high-rate banks of
// the multirate plan).  One CTA = one warp task (group g, stream s); its NCW warps split the time tile into
// chunks of C samples.  Pass 1: warp 0 runs chunk 0 from the true state and writes z at once, warps
// 1..nch-2 run their chunks from zero state without z; the end states meet in shared memory, every warp
// folds s_{c+1} = a1^C s_c + e_c up to its own chunk (a1^C by repeated squaring in double), and pass 2
// reruns chunks 1..nch-1 from their true initial states with z.  Critical path: two chunks instead of
// the whole tile; one launch.
// ---------------------------------------------------------------------------------------------
constexpr int kScanMaxWarps = 16;

// one chunk [cbeg, cbeg + clen) of the staged tile that starts at block sample t0
template <int F, int LPT, bool NOZ>
__device__ __forceinline__ void scan_run_chunk(const float4* __restrict__ win4, const int (&off4)[F], const float4 (&cf)[F],
                                               float2 (&Y)[F], int t0, int cbeg, int clen, int lane, const OutCtx<LPT>& oc)
{
    const int nfull = clen / kBatch;
    const RedCtx rc{};
    float2 Z[kBatch];
    for (int b = 0; b < nfull; ++b) {
        batch_steps<F, true, NOZ>(win4, off4, (cbeg >> 2) + b * (kBatch / 4), cf, Y, Z, kBatch);
        if (!NOZ) emit_batch<LPT, false>(Z, lane, t0 + cbeg + b * kBatch, kBatch, oc, rc, 0);
    }
    const int rem = clen - nfull * kBatch;
    if (rem > 0) {
        batch_steps<F, false, NOZ>(win4, off4, (cbeg >> 2) + nfull * (kBatch / 4), cf, Y, Z, rem);
        if (!NOZ) emit_batch<LPT, false>(Z, lane, t0 + cbeg + nfull * kBatch, rem, oc, rc, 0);
    }
}

template <int F, int LPT>
__global__ void __launch_bounds__(kScanMaxWarps * 32) spiir_filter_scan_kernel(const FilterArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* win = reinterpret_cast<float*>(smem_raw);                   // 4 copies x CS floats
    uint64_t* bar = reinterpret_cast<uint64_t*>(win + 4 * (size_t)a.CS);
    float2* ex = reinterpret_cast<float2*>(win + 4 * (size_t)a.CS + 4);     // [NCW + 1][F][32]: ex[0] = state at the tile start

    const int lane = threadIdx.x & 31, c = threadIdx.x >> 5, NCW = blockDim.x >> 5;
    const int g = blockIdx.x, s = blockIdx.y;
    constexpr int TPG = 32 / LPT;
    const int tl = g * TPG + lane / LPT;
    const bool active = tl < a.T;
    const int t = active ? (a.tmap ? a.tmap[tl] : tl) : 0;
    OutCtx<LPT> oc;
    oc.zt = a.z + ((size_t)s * a.T_rows + t) * (size_t)a.n;
    oc.z_s = a.z + (size_t)s * a.T_rows * (size_t)a.n; oc.n = (size_t)a.n;
    oc.tile = reinterpret_cast<float4*>(ex + (size_t)(NCW + 1) * F * 32) + (size_t)c * (TPG * kTileRow4);
    oc.active = active; oc.acc = a.accumulate != 0; oc.z16 = a.z16 != 0;
    out_ctx_rows<LPT>(oc, a, g, lane);
    const size_t lbase = ((size_t)g * F) * 32 + lane;
    float2* st = a.state + (size_t)s * a.sstride + lbase;

    // coefficient / delay / state loads first: their DRAM round trip overlaps the one of the phase word and the window
    float4 cf[F]; float2 Y[F], Y0[F], aC[F]; int off4[F], dl[F];
#pragma unroll
    for (int f = 0; f < F; ++f) {
        cf[f] = a.coef[lbase + (size_t)f * 32];
        dl[f] = a.dly[lbase + (size_t)f * 32];
        Y[f] = (c == 0) ? st[(size_t)f * 32] : make_float2(0.f, 0.f);
        if (a.apow) aC[f] = a.apow[lbase + (size_t)f * 32];           // a1^C from the plan's table (same chunk length)
    }
    int* sph = reinterpret_cast<int*>(bar + 1);                          // one reader of the phase word per CTA: see filter_body
    uint32_t parity = 0;
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        *sph = phase_parity(a.phase);
        if (a.carry) phase_arrive(a.phase, blockIdx.y * gridDim.x + blockIdx.x, gridDim.x * gridDim.y);
    }
    __syncthreads();
    const int ph = *sph;
    const float* hist_s = a.hbuf[ph] + (size_t)s * a.Dpad;
    const float* x_s = a.x + (size_t)s * a.n;
#pragma unroll
    for (int f = 0; f < F; ++f) {
        const int d = dl[f];
        const int sh = (-d) & 3;
        off4[f] = (sh * a.CS + a.Dpad - d - sh) >> 2;
        if (!a.apow) {
            // a1^C, C = chunk length, by repeated squaring in double (1 us for a 512-thread CTA: only for block lengths
            // the plan holds no table for)
            double pr = 1.0, pi = 0.0, br = (double)cf[f].x, bi = (double)cf[f].y;
            for (int e = a.C; e > 0; e >>= 1) {
                if (e & 1) { const double r = pr * br - pi * bi, q = pr * bi + pi * br; pr = r; pi = q; }
                const double r = br * br - bi * bi, q = 2.0 * br * bi; br = r; bi = q;
            }
            aC[f] = make_float2((float)pr, (float)pi);
        }
    }
    const float4* win4 = reinterpret_cast<const float4*>(win);
    const int ntiles = (a.n + a.NT - 1) / a.NT;
    for (int tile = 0; tile < ntiles; ++tile) {
        const int t0 = tile * a.NT;
        const int len = min(a.NT, a.n - t0);
        __syncthreads();                                               // window and ex[] of the previous tile are free
        stage_window(win, bar, parity, a, hist_s, x_s, t0);
        if (a.carry && ntiles == 1) {
            // carried history for the next block straight from the staged window: W[n + i] is sample n - Dpad + i
            float* hn = a.hbuf[ph ^ 1] + (size_t)s * a.Dpad;
            for (int i = g * blockDim.x + threadIdx.x; i < a.Dpad; i += gridDim.x * blockDim.x) hn[i] = win[a.n + i];
        }
        const int nch = (len + a.C - 1) / a.C;
        const int cbeg = c * a.C, clen = min(a.C, len - cbeg);
        // Phase 1: every chunk but the last runs WITHOUT output to find its end state -- chunk 0 from the true state
        // (so its end is true), the others from zero.  Chunk 0 does not emit yet either: its pass with output is 2x
        // the cost of a pass without, and every other warp would wait for it at the barrier.
        if (c == 0) {
            if (tile > 0) {
#pragma unroll
                for (int f = 0; f < F; ++f) Y[f] = ex[f * 32 + lane];
            }
#pragma unroll
            for (int f = 0; f < F; ++f) Y0[f] = Y[f];
        }
        if (c < nch - 1) {
            if (c > 0) {
#pragma unroll
                for (int f = 0; f < F; ++f) Y[f] = make_float2(0.f, 0.f);
            }
            scan_run_chunk<F, LPT, true>(win4, off4, cf, Y, t0, cbeg, clen, lane, oc);
#pragma unroll
            for (int f = 0; f < F; ++f) ex[((c + 1) * F + f) * 32 + lane] = Y[f];
        }
        __syncthreads();
        // Phase 2: true initial state of every chunk (ex[1] = true end of chunk 0, then y <- a1^C y + zero-state end),
        // and the pass that emits z.
        if (c < nch) {
#pragma unroll
            for (int f = 0; f < F; ++f) {
                float2 v = Y0[f];
                if (c >= 1) {
                    v = ex[(F + f) * 32 + lane];
                    for (int j = 1; j < c; ++j) {
                        const float2 e = ex[((j + 1) * F + f) * 32 + lane];
                        float2 nx;
                        nx.x = fmaf(aC[f].x, v.x, fmaf(-aC[f].y, v.y, e.x));
                        nx.y = fmaf(aC[f].x, v.y, fmaf(aC[f].y, v.x, e.y));
                        v = nx;
                    }
                }
                Y[f] = v;
            }
            scan_run_chunk<F, LPT, false>(win4, off4, cf, Y, t0, cbeg, clen, lane, oc);
            if (c == nch - 1) {
#pragma unroll
                for (int f = 0; f < F; ++f) ex[f * 32 + lane] = Y[f];
            }
        }
    }
    __syncthreads();
    if (c == 0) {
#pragma unroll
        for (int f = 0; f < F; ++f) st[(size_t)f * 32] = ex[f * 32 + lane];
    }
    if (a.carry && ntiles > 1) {
        float* hn = a.hbuf[ph ^ 1] + (size_t)s * a.Dpad;
        for (int i = g * blockDim.x + threadIdx.x; i < a.Dpad; i += gridDim.x * blockDim.x) {
            const int k = a.n - a.Dpad + i;
            hn[i] = (k >= 0) ? x_s[k] : hist_s[a.n + i];
        }
    }
}

// Several banks that share a lane mapping (F, LPT) in one launch: blockIdx.z picks the bank.  Used by the
// multirate plan for its low-rate banks, each of which is only a few microseconds of work.
constexpr int kMaxMulti = 8;
struct MultiFilterArgs {
    FilterArgs bank[kMaxMulti];
    int gx[kMaxMulti], gy[kMaxMulti];
};

template <int F, int LPT>
__global__ void __launch_bounds__(kMaxWarps * 32) spiir_filter_multi_kernel(const __grid_constant__ MultiFilterArgs m)
{
    const int k = blockIdx.z;
    if ((int)blockIdx.x >= m.gx[k] || (int)blockIdx.y >= m.gy[k]) return;
    filter_body<F, LPT, false, false>(m.bank[k], blockIdx.x, blockIdx.y, m.gx[k], m.gy[k]);
}

// ---------------------------------------------------------------------------------------------
// Chunk carry (row a7): per filter, in place over chunk_st[s][c][i]:
//   before: chunk_st[0] = true end state of chunk 0, chunk_st[c>=1] = zero-state end of chunk c
//   after : chunk_st[c] = true INITIAL state of chunk c  (chunk_st[0] = carried state)
// s_{c+1} = a1^C * s_c + e_c.  a1^C by repeated squaring in double.
// ---------------------------------------------------------------------------------------------
__global__ void spiir_chunk_carry_kernel(const float4* __restrict__ coef, const float2* __restrict__ state, size_t sstride,
                                         float2* chunk_st, int nfilt /* G*F*32 */, int S, int NC, int C)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nfilt) return;
    const float4 cf = coef[i];
    double pr = 1.0, pi = 0.0, br = (double)cf.x, bi = (double)cf.y;
    for (int e = C; e > 0; e >>= 1) {
        if (e & 1) { double r = pr * br - pi * bi, q = pr * bi + pi * br; pr = r; pi = q; }
        double r = br * br - bi * bi, q = 2.0 * br * bi; br = r; bi = q;
    }
    const float aCr = (float)pr, aCi = (float)pi;
    for (int s = 0; s < S; ++s) {
        float2* cs = chunk_st + (size_t)s * NC * nfilt + i;
        float2 cur = cs[0];                                // true end of chunk 0 = initial state of chunk 1
        cs[0] = state[(size_t)s * sstride + i];            // initial state of chunk 0
        // the zero-state ends are fetched eight at a time so that their load latencies overlap
        for (int c0 = 1; c0 < NC; c0 += 8) {
            float2 ec[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) ec[j] = c0 + j < NC ? cs[(size_t)(c0 + j) * nfilt] : make_float2(0.f, 0.f);
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                if (c0 + j < NC) {
                    cs[(size_t)(c0 + j) * nfilt] = cur;
                    float2 nxt;
                    nxt.x = fmaf(aCr, cur.x, fmaf(-aCi, cur.y, ec[j].x));
                    nxt.y = fmaf(aCr, cur.y, fmaf(aCi, cur.x, ec[j].y));
                    cur = nxt;
                }
            }
        }
    }
}

// state gather / scatter between plan order and the caller's [S][T][L] order
__global__ void spiir_state_permute_kernel(float2* plan_state, float2* user_state, const int* __restrict__ pos,
                                           size_t TL, size_t nfilt, int S, int to_user)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= TL) return;
    const int p = pos[i];
    for (int s = 0; s < S; ++s) {
        if (to_user) user_state[(size_t)s * TL + i] = plan_state[(size_t)s * nfilt + p];
        else plan_state[(size_t)s * nfilt + p] = user_state[(size_t)s * TL + i];
    }
}

// input history between the plan's ping-pong buffers ([S][Dpad], the newest sample last) and the caller's
// [S][D] (the last D samples, oldest first)
__global__ void spiir_hist_copy_kernel(float* const hbuf0, float* const hbuf1, const int* __restrict__ phase, float* user,
                                       int S, int Dpad, int D, int to_user)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S * Dpad) return;
    const int s = i / Dpad, j = i % Dpad;
    float* cur = (phase_parity(phase) ? hbuf1 : hbuf0) + (size_t)s * Dpad;
    const int k = j - (Dpad - D);                       // index in the caller's row
    if (to_user) { if (k >= 0) user[(size_t)s * D + k] = cur[j]; }
    else cur[j] = k >= 0 ? user[(size_t)s * D + k] : 0.f;
}

}  // namespace spiir
