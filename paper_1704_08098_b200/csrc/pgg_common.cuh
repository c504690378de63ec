// pgg_common.cuh -- argument block shared by all phase-kernel variants, and the
// lattice accessors of the two canonical layouts (include/pgg.h).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "pgg_device.cuh"

namespace pgg {

constexpr int kFmtU8 = 0;
constexpr int kFmtBits = 1;
constexpr int kTableSize = 153;  // 3 values of ds x 51 values of dA
// The game whose payoffs decide the step.  kGamePD is the prisoner's dilemma the paper names as the
// first other game its scheme adapts to (readings G1-G4 in include/pgg.h): its 50
// thresholds, indexed s_x*25 + n_x*5 + n_y, sit at the front of the lattice's 153-entry table slot.
constexpr int kGamePGG = 0;
constexpr int kGamePD = 1;
constexpr int kPdTableSize = 50;

// One phase launch covers B lattices (B = 1 for pgg_sweep).  Per-lattice data
// live in device arrays indexed by the lattice number b.
struct PhaseArgs {
    uint8_t* lats;                // B lattices, contiguous
    unsigned long long lat_bytes; // bytes per lattice (L*L or L*L/8)
    const uint64_t* seeds;        // [B]
    const uint32_t* tables;       // [B][153] acceptance thresholds
    const uint8_t* order;         // [B][order_stride][16] phase classes of this chunk of MCS
    unsigned long long* deltas;   // [B][n_mcs] signed flip sums (two's complement) or nullptr
    uint32_t L;
    uint32_t order_stride;        // MCS per chunk held in `order`
    uint32_t n_mcs;               // row length of `deltas`
    uint32_t t_begin;             // MCS index of deltas[.][0]
};

// ---------------------------------------------------------------------------
// Site accessors with periodic boundaries.  Coordinates may lie
// in [-4, L+4).
// ---------------------------------------------------------------------------
__device__ __forceinline__ int wrap_coord(int a, int L)
{
    a = (a < 0) ? a + L : a;
    return (a >= L) ? a - L : a;
}

template <int FMT>
struct Lattice;

template <>
struct Lattice<kFmtU8> {
    uint8_t* p;
    int L;
    __device__ __forceinline__ int get(int i, int j) const
    {
        return p[(size_t)wrap_coord(i, L) * (size_t)L + (size_t)wrap_coord(j, L)];
    }
    // s(i,j) <- v for an in-range site whose current value is the opposite one
    __device__ __forceinline__ void flip_to(int i, int j, int v) const
    {
        p[(size_t)i * (size_t)L + (size_t)j] = (uint8_t)v;
    }
};

template <>
struct Lattice<kFmtBits> {
    uint8_t* p;
    int L;
    __device__ __forceinline__ int get(int i, int j) const
    {
        const int ii = wrap_coord(i, L), jj = wrap_coord(j, L);
        const uint32_t w = reinterpret_cast<const uint32_t*>(p)[(size_t)ii * (size_t)(L >> 5) +
                                                                (size_t)(jj >> 5)];
        return (int)((w >> (jj & 31)) & 1u);
    }
    // Eight sites of one class share a word, so a flip must be an atomic
    // read-modify-write of its own bit.
    __device__ __forceinline__ void flip_to(int i, int j, int /*v*/) const
    {
        atomicXor(reinterpret_cast<uint32_t*>(p) + (size_t)i * (size_t)(L >> 5) + (size_t)(j >> 5),
                  1u << (j & 31));
    }
};

// Integer payoff kernel A_x = sum over the five groups of x of N(z) (include/pgg.h).
// Expanding the five crosses: the centre is counted 5 times, each nearest and
// each diagonal neighbour twice, each axial distance-2 site once.
template <class Lat>
__device__ __forceinline__ int payoff_A(const Lat& lat, int i, int j)
{
    const int c = lat.get(i, j);
    const int nn = lat.get(i - 1, j) + lat.get(i + 1, j) + lat.get(i, j - 1) + lat.get(i, j + 1);
    const int dg = lat.get(i - 1, j - 1) + lat.get(i - 1, j + 1) + lat.get(i + 1, j - 1) +
                   lat.get(i + 1, j + 1);
    const int ax = lat.get(i - 2, j) + lat.get(i + 2, j) + lat.get(i, j - 2) + lat.get(i, j + 2);
    return 5 * c + 2 * (nn + dg) + ax;
}

// Prisoner's dilemma: number of cooperators among the four nearest neighbours of (i,j) (G3).
template <class Lat>
__device__ __forceinline__ int pd_neighbour_count(const Lat& lat, int i, int j)
{
    return lat.get(i - 1, j) + lat.get(i + 1, j) + lat.get(i, j - 1) + lat.get(i, j + 1);
}

__device__ __forceinline__ int table_index(int dA, int ds)
{
    return (ds + 1) * 51 + (dA + 25);
}

}  // namespace pgg
