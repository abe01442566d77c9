// spiir_resample_tc.cuh -- up-by-2 (+ accumulate) with the 192-tap (or 32-tap) FIR on the 5th-generation tensor cores
// (row a10 of SURVEY.md section 8; Eq. 9).
//
// The polyphase FIR  w[2m+p] = 2 sum_{q<96} h[2q+p] v[m-q]  of a strip of rows is a dense contraction with a banded
// Toeplitz matrix; a strip is 48 complex rows, one tile = 64 input positions -> 128 outputs:
//     D[t, row'] = sum_k T[t, k] * X[row', k]
//   T: 128 outputs of the tile x a window of K = 160 input samples (96 before the tile + its 64 inputs),
//      T[2m'+p, k] = 2 h[2 (96 + m' - k) + p] for 1 <= k - m' <= 96, zero elsewhere (60 % dense).  It is the same for
//      every tile, so it lives in TENSOR MEMORY for the whole kernel (the A operand of tcgen05.mma may come from TMEM);
//   X: 96 real rows (re of the 48 rows, then im) x the window, the DATA, in shared memory (B operand, K-major);
//   D: 128 lanes (outputs) x 96 columns (real rows) of float32 in TMEM, double-buffered (T: 160 + 80 + 80 columns, D: 2 x 96 = all 512 columns).
// tcgen05.mma kind::tf32 (M = 128, N = 96, K = 8 per instruction; measured on this B200: 55 cycles per instruction
// up to N = 64, 67 at N = 128 = the nominal TF32 rate, so narrow tiles waste the pipe).  One TF32 pass has 2^-11
// input precision, far outside the 1e-5 tolerance: every operand is split into a TF32-exact high part and the
// float32 remainder, T X = T_hi X_hi + T_lo X + T X_lo (the dropped T_lo X_lo term is 2^-22 relative).  Only the first
// product needs TF32; the two correction terms are 2^-11 of it, so bf16 operands (2^-9 relative) leave them exact to
// 2^-20: they run as kind::f16 instructions with K = 16 (bf16(T_lo) bf16(X) + bf16(T) bf16(X_lo), 10 + 10 instructions per
// tile instead of 20 + 20 in TF32) into the SAME float32 accumulator.  Measured against the float64 oracle: rel-L2 8.5e-7
// (three TF32 passes: 7.5e-7; the CUDA-core kernel: 1.5e-7).
//
// The data operands use the canonical K-major, non-swizzled layout: 16-byte "units" of 4 consecutive TF32 samples (8
// bf16 samples), unit u of real row r at u * 1536 + r * 16.  Each is a RING of 7 chunks of 32 samples (56 TF32 units,
// 28 bf16 units, twice): a tile's window is 5 consecutive chunks, every tile advances it by two and two chunks are free
// for the loader to run a whole tile ahead; each input sample is written to shared memory once and read by 2.5 tiles; an
// instruction takes two adjacent units and never straddles the ring's end.
//
// The kernel is a template over (HK, R): R = taps per polyphase branch, HK = the window's halo in whole chunks.  <96, 96> is
// the 192-tap filter described above; <32, 16> is the paper's own 32-tap up filter run as a 64-tap filter whose
// outer taps are zero (window of 96 samples, 12 + 6 + 6 instructions per tile): that stage is HBM-bound by its arithmetic,
// but the CUDA-core streaming kernel was held at 55 % of the HBM peak by L1 wavefronts; here it moves data the same way as
// the 192-tap stage and runs at the same 84 %.
//
// Roles (384 threads): one thread of warp 11 fetches the raw chunks (ROWS rows x 32 samples) with TMA tile copies through
// a tensor map of the input into a 4-slot staging ring (48 KB of loads in flight per SM); warps 0-5 read a staged chunk,
// split it into the TF32 high part and the two bf16 correction operands and store them as the data operands; warp 10 issues the MMAs (one thread) and owns
// TMEM; warps 6-9 drain the accumulator (tcgen05.ld): a lane is an output sample, so a warp writes 256 contiguous bytes of
// one row per store -- no transposition; with accumulate the store is a vector reduction (red.global.add.v2.f32) done
// by the L2.  mbarriers: sfull[4] / sempty[4] per staging slot, full[7] / empty[7] per ring chunk, tfull[2] / tempty[2]
// for the accumulator buffers.  CTAs are persistent over (strip, time segment) units.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "spiir_common.cuh"

namespace spiir {
namespace tc {

#ifndef SPIIR_TC_ROWS
#define SPIIR_TC_ROWS 48
#endif
constexpr int ROWS = SPIIR_TC_ROWS;            // complex rows per strip: 48 (double-buffered accumulator); 64 (N = 128) leaves one buffer and measured slower
constexpr int NR = 2 * ROWS;                   // real rows = UMMA N
constexpr int TIN = 64;                        // input samples per tile
constexpr int MOUT = 2 * TIN;                  // outputs per tile = UMMA M
constexpr int CHS = 32;                        // samples per chunk
constexpr int CHU = CHS / 4;                   // units per chunk
constexpr int UNIT_BYTES = NR * 16;
constexpr int STG_SLOTS = 4;                   // raw chunks in flight per CTA (TMA tensor copies, 48 KB)
constexpr int STG_HALF = ROWS * 128;           // half a chunk: ROWS x 16 samples = ROWS x 128 bytes, 128-byte swizzle
constexpr int STG_BYTES = 2 * STG_HALF;
constexpr int LOADER_WARPS = ROWS / 8;         // warps that split and store the data operand
constexpr int LOADERS = LOADER_WARPS * 32;
constexpr int EPI_WARPS = 4;
constexpr int THREADS = (LOADER_WARPS + EPI_WARPS + 2) * 32;   // loader warps, epilogue warps, 1 MMA warp, 1 TMA warp (384 threads at 48 rows)
static_assert(LOADERS == ROWS * CHU / 2, "a loader thread owns 8 consecutive samples of one row of a chunk");
constexpr int TMEM_COLS = 512;

// What depends on the filter: R = taps per polyphase branch (96 for the 192-tap filter of configs[3], 16 for the paper's
// 32-tap up filter), HK >= R = the samples in front of a tile that its window covers, a multiple of the chunk
// length (96 and 32: the 32-tap filter runs as a 64-tap one whose outer taps are zero).
template <int HK, int R>
struct Geo {
    static_assert(HK % CHS == 0 && R <= HK && R >= 1, "window halo = whole chunks");
    static constexpr int KWIN = HK + TIN;               // 160 / 96 samples per window
    static constexpr int KSTEPS = KWIN / 8;             // TF32 k-steps of a tile (bf16: half as many)
    static constexpr int WIN_CH = KWIN / CHS;           // 5 / 3 chunks per window
    static constexpr int HALO_CH = HK / CHS;            // chunks in front of the first tile of a unit
    static constexpr int RING_CH = WIN_CH + 2;          // a whole tile (two chunks) of prefetch space
    static constexpr int RING_UNITS = RING_CH * CHU;    // even
    static constexpr int PART_BYTES = RING_UNITS * UNIT_BYTES;
    static constexpr int OFF_XB = PART_BYTES;           // bf16(x): units of 8 samples, half the bytes of the TF32 part
    static constexpr int OFF_XLB = PART_BYTES + PART_BYTES / 2;   // bf16(x - tf32(x))
    static constexpr int OFF_STG = (2 * PART_BYTES + 1023) / 1024 * 1024;   // the 128-byte swizzle pattern repeats every 1024 bytes
    static constexpr int OFF_BAR = OFF_STG + STG_SLOTS * STG_BYTES;
    static constexpr int NBAR = 2 * RING_CH + 4 + 2 * STG_SLOTS;
    static constexpr int OFF_TPTR = OFF_BAR + NBAR * 8;
    static constexpr int SMEM_BYTES = OFF_TPTR + 16;
    static_assert(STG_HALF % 1024 == 0 && SMEM_BYTES <= 227 * 1024, "shared memory");
    // TMEM columns: T as its TF32 high part, bf16(low part), bf16(T) (two per column); accumulator buffer(s) behind
    static constexpr int COL_THI = 0, COL_TLB = KWIN, COL_TB = KWIN + KWIN / 2, COL_D = 2 * KWIN;
    static constexpr int NBUF = (2 * KWIN + 2 * NR <= TMEM_COLS) ? 2 : 1;
    static constexpr int HIST = R - 1;                  // carried history samples per row
};

struct UpTcArgs {
    const float2* in;        // [rows][n_in]
    float2*       out;       // [rows][2 n_in]
    float2*       hbuf[2];   // [rows][95] ping-pong history
    int*          phase;
    const float*  taps;      // DEVICE: the 192 taps h[j]
    int rows, n_in, accumulate;
    int nstrips, nsegs, seg_tiles, tiles_per_row;
    int in16;                // rows of `in` are 16-byte aligned
};

__device__ __forceinline__ uint32_t s32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void bar_init(uint32_t bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void bar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// Bounded spin: a protocol error becomes a trap (a CUDA error the caller sees), never a hung GPU.
__device__ __forceinline__ void bar_wait(uint32_t bar, uint32_t parity)
{
    for (int it = 0; it < (1 << 28); ++it) {
        uint32_t ok;
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return;
    }
    __trap();
}
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo, uint32_t sbo)
{
    // K-major, no swizzle: start address, leading (K) and stride (8-row group) byte offsets in 16-byte units, version 1
    return (uint64_t)((addr >> 4) & 0x3fff) | ((uint64_t)((lbo >> 4) & 0x3fff) << 16) | ((uint64_t)((sbo >> 4) & 0x3fff) << 32) |
           ((uint64_t)1 << 46);
}
// D[tmem_d] (+)= A[tmem_a] * B[smem descriptor]: the A operand (the Toeplitz matrix) is read from tensor memory
__device__ __forceinline__ void umma_tf32_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n"
                 " tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, {%5, %5, %5, %5}, p;\n}"
                 ::"r"(tmem_d), "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(accumulate), "r"(0u) : "memory");
}
// 32 consecutive columns of this thread's TMEM lane <-> 32 registers
// same with bf16 operands (K = 16 per instruction; A: two elements per TMEM column) accumulating into the same float32 D
__device__ __forceinline__ void umma_bf16_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n"
                 " tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, {%5, %5, %5, %5}, p;\n}"
                 ::"r"(tmem_d), "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(accumulate), "r"(0u) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                 "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
                   "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
                   "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
                 : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                 : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&v)[8])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]) : "r"(taddr));
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&v)[32])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
                 "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};"
                 ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
                   "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]),
                   "r"(v[16]), "r"(v[17]), "r"(v[18]), "r"(v[19]), "r"(v[20]), "r"(v[21]), "r"(v[22]), "r"(v[23]),
                   "r"(v[24]), "r"(v[25]), "r"(v[26]), "r"(v[27]), "r"(v[28]), "r"(v[29]), "r"(v[30]), "r"(v[31]) : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[16])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
                 ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
                   "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
}
// two floats -> packed bf16 pair, `lo` in the low half (= the lower K index)
__device__ __forceinline__ uint32_t bf16x2(float lo, float hi)
{
    const __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<const uint32_t*>(&v);
}
__device__ __forceinline__ void sts128u(uint32_t addr, uint32_t x, uint32_t y, uint32_t z, uint32_t w)
{
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
__device__ __forceinline__ void sts128(uint32_t addr, float4 v)
{
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ float4 lds128(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void bar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// TMA tile copy global -> shared through a 2-D tensor map (box = 32 floats x ROWS rows); completion is counted on the mbarrier
__device__ __forceinline__ void tma_g2s_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ float tf32_hi(float x)
{
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return __uint_as_float(r);
}

// sample m of a row (m relative to the block): history for -95 <= m < 0, zero outside
template <int HIST>
__device__ __forceinline__ float2 sample_at(const float2* in_row, const float2* hist_row, int m, int n_in)
{
    if (m >= 0) return m < n_in ? in_row[m] : make_float2(0.f, 0.f);
    return m >= -HIST ? hist_row[HIST + m] : make_float2(0.f, 0.f);
}


template <int HK, int R>
__global__ void __launch_bounds__(THREADS, 1) spiir_up2_tc_kernel(const UpTcArgs a, const __grid_constant__ CUtensorMap in_map)
{
    using G = Geo<HK, R>;

    extern __shared__ __align__(1024) unsigned char sm[];
    const uint32_t sbase = s32(sm);
    const uint32_t bar0 = sbase + G::OFF_BAR;
    auto full = [&](int i) { return bar0 + 8u * (uint32_t)i; };
    auto empty = [&](int i) { return bar0 + 8u * (uint32_t)(G::RING_CH + i); };
    auto tfull = [&](int i) { return bar0 + 8u * (uint32_t)(2 * G::RING_CH + i); };
    auto tempty = [&](int i) { return bar0 + 8u * (uint32_t)(2 * G::RING_CH + 2 + i); };
    auto sfull = [&](int i) { return bar0 + 8u * (uint32_t)(2 * G::RING_CH + 4 + i); };
    auto sempty = [&](int i) { return bar0 + 8u * (uint32_t)(2 * G::RING_CH + 4 + STG_SLOTS + i); };
    uint32_t* tptr = reinterpret_cast<uint32_t*>(sm + G::OFF_TPTR);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int ph = phase_read(a.phase);
    const float2* hcur = a.hbuf[ph];
    float2* hnext = a.hbuf[ph ^ 1];

    // ---- one-time setup: barriers, tensor memory, the Toeplitz operand into TMEM --------------------------
    if (tid == 0) {
        for (int i = 0; i < G::RING_CH; ++i) { bar_init(full(i), LOADER_WARPS); bar_init(empty(i), 1); }
        for (int i = 0; i < 2; ++i) { bar_init(tfull(i), 1); bar_init(tempty(i), EPI_WARPS); }
        for (int i = 0; i < STG_SLOTS; ++i) { bar_init(sfull(i), 1); bar_init(sempty(i), LOADER_WARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == LOADER_WARPS + EPI_WARPS) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(s32(tptr)), "r"(TMEM_COLS));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tptr;
    {   // lane t of TMEM = output t of a tile.  A warp reaches the TMEM lanes 32 (warp mod 4) .. + 31: the twelve warps share
        // the work as three per lane quarter, each taking every third block of 32 columns (one warp per quarter took 6 us)
        const int t = (warp & 3) * 32 + lane;
        const uint32_t lane_addr = tmem + ((uint32_t)((warp & 3) * 32) << 16);
        // T[t = 2m'+p][k] = 2 h[2 (HK + m' - k) + p] for HK - R < k - m' <= HK, split into a TF32-exact high part and the
        // float32 remainder, computed from the taps (L1-resident) straight into this thread's TMEM lane
        const int mp = t >> 1, pp = t & 1;
        static_assert(THREADS == 384, "three warps per TMEM lane quarter");
        for (int c0 = (warp >> 2) * 32; c0 < G::KWIN; c0 += 3 * 32) {
            uint32_t vh[32], vlb[16], vb[16];
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                float v[2], l[2];
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int dk = c0 + 2 * i + e - mp;
                    v[e] = (dk <= HK && dk > HK - R) ? 2.f * __ldg(a.taps + 2 * (HK - dk) + pp) : 0.f;
                    const float h = tf32_hi(v[e]);
                    vh[2 * i + e] = __float_as_uint(h);
                    l[e] = v[e] - h;
                }
                vlb[i] = bf16x2(l[0], l[1]);
                vb[i] = bf16x2(v[0], v[1]);
            }
            tmem_st32(lane_addr + G::COL_THI + (uint32_t)c0, vh);
            tmem_st16(lane_addr + G::COL_TLB + (uint32_t)(c0 >> 1), vlb);
            tmem_st16(lane_addr + G::COL_TB + (uint32_t)(c0 >> 1), vb);
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");

    const int nunits = a.nstrips * a.nsegs;
    int cbase = 0, tbase = 0, sbase_ch = 0;                            // chunks / tiles / staged chunks of this CTA's earlier units
    for (int u = blockIdx.x; u < nunits; u += gridDim.x) {
        const int strip = u / a.nsegs, seg = u % a.nsegs;
        const int tile0 = seg * a.seg_tiles;
        const int J = min(a.seg_tiles, a.tiles_per_row - tile0);
        const int ms = tile0 * TIN;
        const int row0 = strip * ROWS;
        const int nch = G::WIN_CH - 2 + 2 * J;                            // chunks of this unit: 3 of halo + 2 per tile

        // A chunk that lies inside the block with 16-byte aligned rows is STAGED: one thread fetches its raw samples with
        // two TMA tile copies (ROWS rows x 16 samples each, through the tensor map of `in`) into a ring of STG_SLOTS slots,
        // so STG_SLOTS chunks of DRAM latency are in flight whatever the loader warps are doing.  (Loads prefetched in
        // registers were not: ptxas gave every prefetch batch the same scoreboard, so waiting for the oldest batch waited
        // for the newest; one bulk copy per row was no better: the TMA unit took ~70 cycles per 256-byte request.)
        // Other chunks (history in front of the block, ragged end, unaligned rows) are read element by element.
        auto staged = [&](int ci) {
            const int mc = ms - HK + ci * CHS;
            return a.in16 && mc >= 0 && mc + CHS <= a.n_in;
        };
        if (warp < LOADER_WARPS) {
            // ===== loaders: split a chunk (ROWS x 32 samples) into TF32 high / low parts and store it as the MMA's data operand.
            // Thread item = (row r, unit u): 4 consecutive samples of one row = two 16-byte reads from the staging slot
            // (consecutive lanes = consecutive rows; the 128-byte swizzle puts piece j of row r at j ^ (r mod 8):
            // conflict-free) and, after the split, four 16-byte stores (re / im, high / low; consecutive lanes =
            // consecutive 16-byte slots of one unit: conflict-free). =====
            const int hfirst = a.n_in - G::HIST;                     // first block sample that is part of the next history
            // Carried history of this strip's rows = the last 95 samples of (history ++ block).  A block of at least 95 samples
            // supplies all of them, and they pass through the loaders' registers anyway (written below); shorter blocks
            // take this explicit copy.
            if (seg == 0 && hfirst < 0) {
                for (int i = tid; i < ROWS * G::HIST; i += LOADERS) {
                    const int rr = i / G::HIST, k = i % G::HIST, rw = row0 + rr;
                    if (rw < a.rows) {
                        const int g = a.n_in - G::HIST + k;
                        hnext[(size_t)rw * G::HIST + k] =
                            g >= 0 ? a.in[(size_t)rw * a.n_in + g] : hcur[(size_t)rw * G::HIST + a.n_in + k];
                    }
                }
            }
            int sc = sbase_ch;
            for (int ci = 0; ci < nch; ++ci) {
                const int c = cbase + ci, slot = c % G::RING_CH, fill = c / G::RING_CH;
                const int mc = ms - HK + ci * CHS;                    // first sample of the chunk
                const bool stg = staged(ci);
                const int ss = sc % STG_SLOTS;
                constexpr int ITEMS = 2;                                // two units of 4 samples: 8 consecutive samples of row r
                const int r = tid % ROWS, up = tid / ROWS;              // up: which 8 samples of the chunk (0 .. 3)
                float4 v[ITEMS][2];                                     // (re, im) of samples 4u .. 4u + 3, u = 2 up + k
                if (stg) {
                    bar_wait(sfull(ss), (uint32_t)((sc / STG_SLOTS) & 1));
#pragma unroll
                    for (int k = 0; k < ITEMS; ++k) {
                        const int u = 2 * up + k;
                        const uint32_t src = sbase + G::OFF_STG + (uint32_t)(ss * STG_BYTES + (u >> 2) * STG_HALF + r * 128);
                        const int j = 2 * (u & 3), x = r & 7;
                        v[k][0] = lds128(src + (uint32_t)((j ^ x) << 4));
                        v[k][1] = lds128(src + (uint32_t)(((j + 1) ^ x) << 4));
                    }
                    __syncwarp();
                    if (lane == 0) bar_arrive(sempty(ss));              // the slot may be refilled
                    ++sc;
                } else {
#pragma unroll
                    for (int k = 0; k < ITEMS; ++k) {
                        const int u = 2 * up + k;
                        const int row = row0 + r, m = mc + 4 * u;
                        float2 q[4];
#pragma unroll
                        for (int e = 0; e < 4; ++e) q[e] = make_float2(0.f, 0.f);
                        if (row < a.rows) {
                            const float2* in_row = a.in + (size_t)row * a.n_in;
                            const float2* hist_row = hcur + (size_t)row * G::HIST;
#pragma unroll
                            for (int e = 0; e < 4; ++e) q[e] = sample_at<G::HIST>(in_row, hist_row, m + e, a.n_in);
                        }
                        v[k][0] = make_float4(q[0].x, q[0].y, q[1].x, q[1].y);
                        v[k][1] = make_float4(q[2].x, q[2].y, q[3].x, q[3].y);
                    }
                }
                // the next history = the block's last 95 samples: written by the unit that owns them (not from a halo)
                if (ci >= G::HALO_CH && hfirst >= 0 && mc + CHS > hfirst) {
#pragma unroll
                    for (int k = 0; k < ITEMS; ++k) {
                        const int u = 2 * up + k;
                        const int row = row0 + r, g = mc + 4 * u - hfirst;
                        if (row < a.rows) {
                            float2* hrow = hnext + (size_t)row * G::HIST;
                            const float2 q[4] = {make_float2(v[k][0].x, v[k][0].y), make_float2(v[k][0].z, v[k][0].w),
                                                 make_float2(v[k][1].x, v[k][1].y), make_float2(v[k][1].z, v[k][1].w)};
#pragma unroll
                            for (int e = 0; e < 4; ++e)
                                if (g + e >= 0 && g + e < G::HIST && mc + 4 * u + e < a.n_in) hrow[g + e] = q[e];
                        }
                    }
                }
                if (fill > 0) bar_wait(empty(slot), (uint32_t)((fill - 1) & 1));
                uint32_t bre[4], bim[4], lre[4], lim[4];                // bf16 pairs of x and of x - tf32(x)
#pragma unroll
                for (int k = 0; k < ITEMS; ++k) {
                    const int u = 2 * up + k;
                    const float4 wre = make_float4(v[k][0].x, v[k][0].z, v[k][1].x, v[k][1].z);
                    const float4 wim = make_float4(v[k][0].y, v[k][0].w, v[k][1].y, v[k][1].w);
                    const float4 hre = make_float4(tf32_hi(wre.x), tf32_hi(wre.y), tf32_hi(wre.z), tf32_hi(wre.w));
                    const float4 him = make_float4(tf32_hi(wim.x), tf32_hi(wim.y), tf32_hi(wim.z), tf32_hi(wim.w));
                    const uint32_t addr = sbase + (uint32_t)(slot * CHU + u) * UNIT_BYTES + (uint32_t)r * 16;
                    sts128(addr, hre);
                    sts128(addr + ROWS * 16, him);
                    bre[2 * k] = bf16x2(wre.x, wre.y); bre[2 * k + 1] = bf16x2(wre.z, wre.w);
                    bim[2 * k] = bf16x2(wim.x, wim.y); bim[2 * k + 1] = bf16x2(wim.z, wim.w);
                    lre[2 * k] = bf16x2(wre.x - hre.x, wre.y - hre.y); lre[2 * k + 1] = bf16x2(wre.z - hre.z, wre.w - hre.w);
                    lim[2 * k] = bf16x2(wim.x - him.x, wim.y - him.y); lim[2 * k + 1] = bf16x2(wim.z - him.z, wim.w - him.w);
                }
                {
                    const uint32_t addr = sbase + (uint32_t)(slot * (CHU / 2) + up) * UNIT_BYTES + (uint32_t)r * 16;
                    sts128u(addr + G::OFF_XB, bre[0], bre[1], bre[2], bre[3]);
                    sts128u(addr + G::OFF_XB + ROWS * 16, bim[0], bim[1], bim[2], bim[3]);
                    sts128u(addr + G::OFF_XLB, lre[0], lre[1], lre[2], lre[3]);
                    sts128u(addr + G::OFF_XLB + ROWS * 16, lim[0], lim[1], lim[2], lim[3]);
                }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                __syncwarp();
                if (lane == 0) bar_arrive(full(slot));                  // one arrival per warp
            }
        } else
        if (warp == LOADER_WARPS + EPI_WARPS + 1) {
            // ===== copy thread: two tile copies per staged chunk, up to STG_SLOTS chunks ahead of the loaders.  Rows past the
            // end of the batch are zero-filled by the TMA unit (and count in the transaction bytes). =====
            if (lane == 0) {
                int sc = sbase_ch;
                for (int ci = 0; ci < nch; ++ci) {
                    if (!staged(ci)) continue;
                    const int ss = sc % STG_SLOTS, f = sc / STG_SLOTS;
                    if (f > 0) bar_wait(sempty(ss), (uint32_t)((f - 1) & 1));
                    bar_expect_tx(sfull(ss), (uint32_t)STG_BYTES);
                    const int c0 = 2 * (ms - HK + ci * CHS);          // float index of the chunk's first sample
                    const uint32_t dst = sbase + G::OFF_STG + (uint32_t)(ss * STG_BYTES);
                    tma_g2s_2d(dst, &in_map, c0, row0, sfull(ss));
                    tma_g2s_2d(dst + STG_HALF, &in_map, c0 + 32, row0, sfull(ss));
                    ++sc;
                }
            }
            __syncwarp();
        } else
        if (warp == LOADER_WARPS + EPI_WARPS) {
            // ===== MMA issuer (one thread) =====
            if (lane == 0) {
                const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(NR >> 3) << 17) | ((uint32_t)(MOUT >> 4) << 24);
                const uint32_t idesc_bf = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(NR >> 3) << 17) | ((uint32_t)(MOUT >> 4) << 24);
                for (int j = 0; j < J; ++j) {
                    const int cn = cbase + 2 * j + G::WIN_CH - 1;          // newest chunk of this tile's window
                    bar_wait(full(cn % G::RING_CH), (uint32_t)((cn / G::RING_CH) & 1));
                    const int t = tbase + j, buf = t % G::NBUF, use = t / G::NBUF;
                    if (use > 0) bar_wait(tempty(buf), (uint32_t)((use - 1) & 1));   // this buffer's previous tile has been drained
                    const uint32_t d = tmem + G::COL_D + (uint32_t)(buf * NR);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const int wu0 = ((cbase + 2 * j) % G::RING_CH) * CHU;  // ring unit of the window's first unit
                    // T_hi X_hi in TF32 (20 instructions of K = 8), then the two correction terms bf16(T_lo) bf16(X) and
                    // bf16(T) bf16(X_lo) with bf16 operands (10 + 10 instructions of K = 16) into the same accumulator
#pragma unroll 2
                    for (int ks = 0; ks < G::KSTEPS; ++ks) {
                        int ru = wu0 + 2 * ks;
                        if (ru >= G::RING_UNITS) ru -= G::RING_UNITS;
                        umma_tf32_ts(d, tmem + G::COL_THI + (uint32_t)(8 * ks), smem_desc(sbase + (uint32_t)ru * UNIT_BYTES, UNIT_BYTES, 128),
                                     idesc, ks > 0 ? 1u : 0u);
                    }
#pragma unroll 2
                    for (int ks = 0; ks < G::KSTEPS / 2; ++ks) {
                        int ru = (wu0 >> 1) + 2 * ks;                   // units of 8 samples
                        if (ru >= G::RING_UNITS / 2) ru -= G::RING_UNITS / 2;
                        const uint32_t xb = sbase + (uint32_t)ru * UNIT_BYTES;
                        umma_bf16_ts(d, tmem + G::COL_TLB + (uint32_t)(8 * ks), smem_desc(xb + G::OFF_XB, UNIT_BYTES, 128), idesc_bf, 1u);
                        umma_bf16_ts(d, tmem + G::COL_TB + (uint32_t)(8 * ks), smem_desc(xb + G::OFF_XLB, UNIT_BYTES, 128), idesc_bf, 1u);
                    }
                    umma_commit(empty((cbase + 2 * j) % G::RING_CH));     // the window's two oldest chunks are free once these MMAs are done
                    umma_commit(empty((cbase + 2 * j + 1) % G::RING_CH));
                    umma_commit(tfull(buf));
                }
                for (int i = 0; i < G::HALO_CH; ++i) umma_commit(empty((cbase + 2 * J + i) % G::RING_CH));
            }
            __syncwarp();
        } else {
            // ===== epilogue, 128 threads: TMEM lane = output sample, columns = real rows (re of row i in column i, im in
            // column ROWS + i).  The thread drains its whole accumulator row into registers, releases the buffer at once
            // (the next-but-one tile's MMAs may overwrite it) and then stores: a warp writes 256 contiguous bytes of one
            // output row per instruction, no transposition. =====
            const int ew = warp & 3;
            const int tl = ew * 32 + lane;                              // output index within the tile
            for (int j = 0; j < J; ++j) {
                const int t = tbase + j, buf = t % G::NBUF, use = t / G::NBUF;
                const int m0 = ms + j * TIN;
                const bool tok = tl < 2 * min(TIN, a.n_in - m0);
                float2* obase = a.out + (size_t)row0 * 2 * a.n_in + 2 * m0 + tl;
                const uint32_t taddr = tmem + ((uint32_t)(ew * 32) << 16) + G::COL_D + (uint32_t)(buf * NR);
                bar_wait(tfull(buf), (uint32_t)(use & 1));
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                // drain in two halves (ROWS registers each); the buffer is released right after the second drain
#pragma unroll
                for (int h2 = 0; h2 < 2; ++h2) {
                    constexpr int RH = ROWS / 2;                        // rows per half (multiple of 8)
                    uint32_t vre[RH], vim[RH];
#pragma unroll
                    for (int q8 = 0; q8 < RH / 8; ++q8) {
                        tmem_ld8(taddr + RH * h2 + 8 * q8, *reinterpret_cast<uint32_t (*)[8]>(&vre[8 * q8]));
                        tmem_ld8(taddr + ROWS + RH * h2 + 8 * q8, *reinterpret_cast<uint32_t (*)[8]>(&vim[8 * q8]));
                    }
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    if (h2 == 1) {
                        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                        __syncwarp();
                        if (lane == 0) bar_arrive(tempty(buf));
                    }
                    // accumulate = a vector reduction performed by the L2 (one addend per element and call: deterministic);
                    // no read-modify-write round trip through this thread's registers
                    float2* ob = obase + (size_t)(RH * h2) * 2 * a.n_in;
                    const int rbase = row0 + RH * h2;
                    if (a.accumulate) {
#pragma unroll
                        for (int i = 0; i < RH; ++i)
                            if (tok && rbase + i < a.rows)
                                asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(ob + (size_t)i * 2 * a.n_in),
                                             "f"(__uint_as_float(vre[i])), "f"(__uint_as_float(vim[i])) : "memory");
                    } else {
#pragma unroll
                        for (int i = 0; i < RH; ++i)
                            if (tok && rbase + i < a.rows)
                                ob[(size_t)i * 2 * a.n_in] = make_float2(__uint_as_float(vre[i]), __uint_as_float(vim[i]));
                    }
                }
            }
        }
        for (int ci = 0; ci < nch; ++ci) sbase_ch += staged(ci) ? 1 : 0;
        cbase += nch;
        tbase += J;
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    const bool last = last_cta_arrives(a.phase, gridDim.x);           // __syncthreads inside
    if (last) a.phase[0] = ph ^ 1;
    if (warp == LOADER_WARPS + EPI_WARPS) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(TMEM_COLS));
}

}  // namespace tc
}  // namespace spiir
