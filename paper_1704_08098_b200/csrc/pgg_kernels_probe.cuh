// pgg_kernels_probe.cuh -- the ALU ceiling probe of SURVEY 8(d)(ii): "a Philox-only kernel's
// site-draws/s".  Every thread makes `iters` x 2 STEP draws with the shipping step_draw()
// (pgg_device.cuh: Philox4x32-10 with the hoisted round keys, words x0 and x1), two independent
// chains per thread as the phase kernels run them, and xors the results into one word that it
// stores, so nothing is eliminated.  No lattice, no shared memory, no divergence: the rate this
// kernel reaches is the most elementary steps per second any phase kernel could draw for.
#pragma once
#include "pgg_device.cuh"

namespace pgg {

constexpr int kProbeThreads = 256;

__global__ void __launch_bounds__(kProbeThreads, 4)
draw_ceiling_kernel(StepKey sk, uint32_t iters, uint32_t* __restrict__ sink)
{
    const uint32_t tid = blockIdx.x * kProbeThreads + threadIdx.x;
    const uint32_t stride = gridDim.x * kProbeThreads * 2u;
    uint32_t site = 2u * tid, acc = 0u;
    for (uint32_t i = 0; i < iters; ++i) {
        uint32_t a0, a1, b0, b1;
        step_draw(sk, site, a0, a1);
        step_draw(sk, site + 1u, b0, b1);
        acc ^= a0 ^ a1 ^ b0 ^ b1;
        site += stride;
    }
    sink[tid] = acc;
}

}  // namespace pgg
