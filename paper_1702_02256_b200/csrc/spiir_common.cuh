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

}  // namespace spiir
