// pgg_kernels_probe.cuh -- the ALU ceiling probe of SURVEY 8(d)(ii): "a Philox-only kernel's
// site-draws/s".  Every thread makes `iters` x 2 STEP draws with the shipping step_draw()
// (pgg_device.cuh: Philox4x32-10 with the hoisted round keys, words x0 and x1), two independent
// chains per thread as the phase kernels run them, and xors the results into one word that it
// stores, so nothing is eliminated.  No lattice, no shared memory, no divergence: the rate this
// kernel reaches is the most elementary steps per second any phase kernel could draw for.
#pragma once
#include "pgg_common.cuh"

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

// The draw fraction of a state (S9): the number of sites with at least one nearest neighbour of
// the other strategy -- exactly the sites for which an elementary step needs its
// random draw; for all others no draw can change anything.  One thread per site, plain loads.
template <int FMT>
__global__ void __launch_bounds__(256)
interface_count_kernel(const uint8_t* __restrict__ lat_p, uint32_t L, unsigned long long* __restrict__ out)
{
    const Lattice<FMT> lat{const_cast<uint8_t*>(lat_p), (int)L};
    const uint32_t n = L * L;
    unsigned int acc = 0;
    for (uint32_t site = blockIdx.x * blockDim.x + threadIdx.x; site < n; site += gridDim.x * blockDim.x) {
        const int i = (int)(site / L), j = (int)(site - (uint32_t)i * L);
        const int s = lat.get(i, j);
        acc += (lat.get(i - 1, j) != s || lat.get(i + 1, j) != s || lat.get(i, j - 1) != s || lat.get(i, j + 1) != s) ? 1u : 0u;
    }
    acc = __reduce_add_sync(0xFFFFFFFFu, acc);
    if ((threadIdx.x & 31) == 0 && acc) atomicAdd(out, (unsigned long long)acc);
}

}  // namespace pgg
