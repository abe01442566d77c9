// spiir_common.cuh -- device helpers shared by the filter and the resampling kernels.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace spiir {

// ---------------------------------------------------------------------------------------------
// Ping-pong phase kept on the device.  A kernel reads w[0] when it starts; the CTA that finishes last
// (arrival counter w[1]) flips it, so no CTA can observe the flip of its own launch.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int phase_read(const int* w) { return *reinterpret_cast<const volatile int*>(w) & 1; }
__device__ __forceinline__ bool last_cta_arrives(int* w, int total_ctas)
{
    __syncthreads();
    bool last = false;
    // No fence: nothing written by this launch is read before the launch has ended (the flipped phase and the
    // history it points to are consumed by the NEXT launch); a fence would wait for the CTA's SNR stores to drain.
    if (threadIdx.x == 0) {
        last = atomicAdd(w + 1, 1) == total_ctas - 1;
        if (last) w[1] = 0;
    }
    return last;                                     // meaningful in thread 0 only
}


// The same without any wait (filter kernels): w[1] counts kPhaseUnit per finished launch -- every CTA of a launch adds its
// share with a fire-and-forget reduction, in any order and at any time after it has read the word -- and the phase is the
// parity of the number of finished launches, w[1] / kPhaseUnit.  A CTA that reads the word while its own launch is
// under way sees a partial sum below the next multiple, i.e. still the phase the launch started with.  The shares of one
// launch add up to kPhaseUnit whatever its grid, so calls with different block lengths can follow one another.
// ONE thread per CTA reads the word and then adds (same address: program order holds) and hands the value to the others
// through shared memory; threads that each read the word themselves may read it after the CTA's own share and the last
// share of the launch have landed.
constexpr int kPhaseUnit = 1 << 16;                 // grids of up to 65536 CTAs; 2^32 is a multiple, so wrap-around is harmless
__device__ __forceinline__ int phase_parity(const int* w)
{
    return (int)((*reinterpret_cast<const volatile unsigned*>(w + 1) >> 16) & 1u);
}
__device__ __forceinline__ void phase_arrive(int* w, int cta, int total_ctas)      // call from ONE thread per CTA
{
    const int share = kPhaseUnit / total_ctas + (cta == 0 ? kPhaseUnit % total_ctas : 0);
    atomicAdd(reinterpret_cast<unsigned*>(w + 1), (unsigned)share);                 // result unused: compiles to RED
}

}  // namespace spiir
