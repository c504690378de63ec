// pgg_device.cuh -- device-side building blocks shared by the phase kernels:
// Philox4x32-10, the integer payoff kernel A_x and small reductions.
// Product code: shares nothing with oracle/ (the oracle has its own Philox,
// its own table and its own payoff sums).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace pgg {

// Counter tags: word c3 of the Philox counter.
constexpr uint32_t kTagInit = 1u;
constexpr uint32_t kTagOrder = 2u;
constexpr uint32_t kTagStep = 3u;

constexpr uint32_t kPhiloxM0 = 0xD2511F53u;
constexpr uint32_t kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u;
constexpr uint32_t kPhiloxW1 = 0xBB67AE85u;

// Philox4x32-10 (Salmon et al., SC'11), all four output words.  The paper only
// says "random"; north_star fixes the generator, S5 the rounds.
__host__ __device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2,
                                                       uint32_t c3, uint32_t k0, uint32_t k1,
                                                       uint32_t out[4])
{
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)kPhiloxM0 * c0;
        const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += kPhiloxW0;
        k1 += kPhiloxW1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// The per-launch constant part of the STEP draw: the counter is
// (site, t, (k<<8)|c, kTagStep), so only c0 varies inside a launch.  Round 1's
// second product (M1 * c2) and the ten round keys are the same for every site:
// compute them once per launch on the host and pass them by value.
struct StepKey {
    uint32_t k0[10];   // round keys, word 0
    uint32_t k1[10];   // round keys, word 1
    uint32_t r1_c0;    // after round 1: c0 = hi(M1*c2) ^ c1 ^ k0[0]      (site independent)
    uint32_t r1_c1;    // after round 1: c1 = lo(M1*c2)                   (site independent)
    uint32_t r1_x2;    // after round 1: c2 = hi(M0*site) ^ (c3 ^ k1[0]); this is c3 ^ k1[0]
};

__host__ __device__ inline StepKey make_step_key(uint64_t seed, uint32_t t, uint32_t k,
                                                 uint32_t cls)
{
    StepKey s;
    uint32_t a = (uint32_t)(seed & 0xFFFFFFFFu), b = (uint32_t)(seed >> 32);
    for (int i = 0; i < 10; ++i) {
        s.k0[i] = a;
        s.k1[i] = b;
        a += kPhiloxW0;
        b += kPhiloxW1;
    }
    const uint32_t c2 = (k << 8) | cls;
    const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
    s.r1_c0 = (uint32_t)(p1 >> 32) ^ t ^ s.k0[0];
    s.r1_c1 = (uint32_t)p1;
    s.r1_x2 = kTagStep ^ s.k1[0];
    return s;
}

// Words x0 (direction = x0 >> 30) and x1 (uniform u) of the STEP draw of `site`.
// Same function as philox4x32_10 on (site, t, c2, 3): round 1 uses the
// precomputed site-independent half, round 10 skips the product whose result
// only feeds x2, x3.
__device__ __forceinline__ void step_draw(const StepKey& sk, uint32_t site, uint32_t& x0,
                                          uint32_t& x1)
{
    // round 1
    const uint64_t q0 = (uint64_t)kPhiloxM0 * site;
    uint32_t c0 = sk.r1_c0;
    uint32_t c1 = sk.r1_c1;
    uint32_t c2 = (uint32_t)(q0 >> 32) ^ sk.r1_x2;
    uint32_t c3 = (uint32_t)q0;
#pragma unroll
    for (int round = 1; round < 9; ++round) {
        const uint64_t p0 = (uint64_t)kPhiloxM0 * c0;
        const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ sk.k0[round];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ sk.k1[round];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    // round 10: only x0 = hi(M1*c2) ^ c1 ^ k0[9] and x1 = lo(M1*c2) are used
    const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
    x0 = (uint32_t)(p1 >> 32) ^ c1 ^ sk.k0[9];
    x1 = (uint32_t)p1;
}

__device__ __forceinline__ int warp_sum(int v)
{
    return __reduce_add_sync(0xFFFFFFFFu, v);
}

}  // namespace pgg
