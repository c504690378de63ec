// pgg_stencil_lut.cuh -- the payoff stencil A_x - A_y (a5) on bit-packed rows by table lookup; used by the
// kernels that keep the lattice as bits on chip (LEAN, CLUSTER, RESIDENT).
#pragma once
#include <cstdint>

namespace pgg {

// ---------------------------------------------------------------------------
// The payoff stencil on bit rows by table (a5).  A_x - A_y is a signed sum over 12 neighbours of x
// (ring_stencil: offsets a e + b f, e = step towards y, f = the perpendicular step) plus 3 (2 s_x - 1).
// The 12 sites lie in six rows -- a = -2 .. 3 for a vertical e, b = -2 .. 2 (and a spare) for a horizontal
// e -- and, in every row, in the seven columns col(x) - 3 .. col(x) + 3.  So per row: the 7-bit window
// (two word loads, a funnel shift, a mask) indexes a 128-entry table that holds the row's weighted sum:
// six table reads replace fourteen single-bit reads (5 instructions each).  Sites within 3 columns of a
// row end keep the wrapping path (ring_stencil_fr).
//   lut[dir][slot][window] : int8, 4 x 6 x 128 = 3072 bytes, copied to shared memory by every CTA
//   slot s of dir: ring row of x + (s - 2) * step(dir),  step = -1 row for dir 0 (e points up), else +1 row
// ---------------------------------------------------------------------------
struct StencilLut {
    int8_t v[4 * 6 * 128];
};
constexpr int kStencilLutBytes = 4 * 6 * 128;
static_assert(sizeof(StencilLut) == kStencilLutBytes, "StencilLut size");

constexpr StencilLut make_stencil_lut()
{
    StencilLut t{};
    // (a, b, weight): x's 13-site weights minus y's, y = x + e, without the centre pair (include/pgg.h)
    const int term[12][3] = {{-2, 0, 1}, {-1, 0, 1}, {2, 0, -1}, {3, 0, -1}, {-1, 1, 2}, {-1, -1, 2},
                             {2, 1, -2}, {2, -1, -2}, {0, 2, 1}, {0, -2, 1}, {1, 2, -1}, {1, -2, -1}};
    for (int dir = 0; dir < 4; ++dir) {
        // e = (er, ec), f = (fr, fc) in (rows, columns): the directions of SURVEY 8(c) D6 and eoff[4..7]
        const int er = dir == 0 ? -1 : dir == 1 ? 1 : 0, ec = dir == 2 ? -1 : dir == 3 ? 1 : 0;
        const int fr = dir < 2 ? 0 : 1, fc = dir < 2 ? 1 : 0;
        const int step = dir == 0 ? -1 : 1;  // rows per slot
        for (int q = 0; q < 12; ++q) {
            const int dr = term[q][0] * er + term[q][1] * fr, dc = term[q][0] * ec + term[q][1] * fc;
            const int slot = dr * step + 2;  // dr = (slot - 2) * step
            for (int w = 0; w < 128; ++w)
                if ((w >> (dc + 3)) & 1) t.v[(dir * 6 + slot) * 128 + w] += (int8_t)term[q][2];
        }
    }
    return t;
}
__device__ const StencilLut g_stencil_lut = make_stencil_lut();

// lut = the table in shared memory; words = ring0 as 32-bit words; wpr = words per ring row.
// Needs 3 <= col(x) <= L - 4 (the window stays inside the row); the word after the window's first is
// read even when the window does not reach it (the ring is followed by the queues: a valid address).
__device__ __forceinline__ int bits_stencil_lut(int soff, uint32_t dir, int sx, const uint32_t* words, int wpr, const int8_t* lut)
{
    const int base = soff - 3;
    const uint32_t sh = (uint32_t)base & 31u;
    const int stepw = dir == 0u ? -wpr : wpr;
    const uint32_t* p = words + (base >> 5) - 2 * stepw;
    const int8_t* l = lut + dir * 768u;
    int dA = 3 * (2 * sx - 1);
#pragma unroll
    for (int s = 0; s < 6; ++s, p += stepw)
        dA += l[s * 128 + (__funnelshift_r(p[0], p[1], sh) & 127u)];
    return dA;
}

}  // namespace pgg
