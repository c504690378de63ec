// pgg_kernels_dtile.cuh -- the paper's own parallel schedule, the double tiling
// decomposition (Fig. 2, Fig. 3), as PGG_ORDER_DTILE.
//
// Schedule (include/pgg.h, DESIGN.md section 2 readings T1-T4): the lattice is cut
// into 4x4 domains; domain (I,J) = (i>>2, j>>2) has type 2*(I&1) + (J&1) (the
// paper's types 1..4), L % 8 == 0.  One MCS = four parts, the types
// in turn; in a part every domain of the type makes 16 sequential
// elementary steps on its own sites, pick p of domain d = I*(L/4)+J
// in MCS t drawing Philox(ctr = (d, t, p, 5)): focal site = domain row x0>>30,
// column (x0>>28)&3, direction x2>>30, u = x1.
//
// Kernel: one thread per domain of the active type -- the paper's "each thread
// being assigned to one domain" -- but where the paper copies the
// 10x10 patch of Fig. 3 (domain + "three lines outward") into a
// shared-memory block per thread, here the patch is 120 bits in two 64-bit
// registers (10 rows x 12 columns, columns 4J-4 .. 4J+7): staged with 30 aligned
// word loads (uint8) or 10-20 (bit-packed), every one of the 16 picks then runs
// on registers only, flips toggle a register bit, and the 4x4 domain is written
// back once, only if it changed.  A domain whose 6x6 neighbourhood is uniform
// cannot change (S9) and skips its 16 draws.  Race-free in place: same-type
// domains are separated by 4 sites, reads reach 3.
// The flip count of the part is reduced per CTA into deltas[m] (a8).
#pragma once
#include "pgg_common.cuh"

namespace pgg {

constexpr uint32_t kTagDtile = 5u;
constexpr int kDtileThreads = 256;

struct DtilePatch {
    unsigned long long lo, hi;  // rows 0-4 / 5-9 of the patch, 12 bits each
    __device__ __forceinline__ int get(int pr, int pc) const
    {
        const unsigned long long v = pr < 5 ? lo : hi;
        const int sh = 12 * (pr < 5 ? pr : pr - 5) + pc;
        return (int)((v >> sh) & 1ull);
    }
    __device__ __forceinline__ void toggle(int pr, int pc)
    {
        const unsigned long long bit = 1ull << (12 * (pr < 5 ? pr : pr - 5) + pc);
        if (pr < 5) lo ^= bit; else hi ^= bit;
    }
    // A of the site at (pr, pc): 5 s + 2 (nearest + diagonal) + axial distance-2 (include/pgg.h)
    __device__ __forceinline__ int A(int pr, int pc) const
    {
        const int nn = get(pr - 1, pc) + get(pr + 1, pc) + get(pr, pc - 1) + get(pr, pc + 1);
        const int dg = get(pr - 1, pc - 1) + get(pr - 1, pc + 1) + get(pr + 1, pc - 1) + get(pr + 1, pc + 1);
        const int ax = get(pr - 2, pc) + get(pr + 2, pc) + get(pr, pc - 2) + get(pr, pc + 2);
        return 5 * get(pr, pc) + 2 * (nn + dg) + ax;
    }
};

// The 12 sites of lattice row i starting at column c0 (a multiple of 4, may be -4), periodic,
// as 12 bits (bit n = site c0 + n).
template <int FMT>
__device__ __forceinline__ uint32_t dtile_row12(const uint8_t* __restrict__ lat, int L, int i, int c0)
{
    const int ii = wrap_coord(i, L);
    if (FMT == kFmtU8) {
        const uint32_t* row = reinterpret_cast<const uint32_t*>(lat + (size_t)ii * (size_t)L);
        uint32_t out = 0;
#pragma unroll
        for (int w = 0; w < 3; ++w) {
            const uint32_t v = row[wrap_coord(c0 + 4 * w, L) >> 2];
            out |= ((((v & 0x01010101u) * 0x01020408u) >> 24) & 0xFu) << (4 * w);  // bit 0 of each byte
        }
        return out;
    } else {
        const uint32_t* row = reinterpret_cast<const uint32_t*>(lat) + (size_t)ii * (size_t)(L >> 5);
        const int c = wrap_coord(c0, L), o = c & 31;
        const uint32_t w0 = row[c >> 5];
        const uint32_t w1 = o > 20 ? row[wrap_coord(c + 12, L) >> 5] : 0u;  // the field straddles two words
        return __funnelshift_r(w0, w1, o) & 0xFFFu;
    }
}

template <int FMT>
__global__ void __launch_bounds__(kDtileThreads)
dtile_part_kernel(PhaseArgs a, uint32_t m, uint32_t q)
{
    const uint32_t b = blockIdx.y;
    const int L = (int)a.L, M = L >> 2, Mh = M >> 1;
    uint8_t* lat = a.lats + (size_t)b * a.lat_bytes;
    const uint32_t* __restrict__ table = a.tables + (size_t)b * kTableSize;
    const uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x;
    int delta = 0;
    if (idx < (uint32_t)Mh * (uint32_t)Mh) {
        const int Ih = (int)(idx / (uint32_t)Mh), Jh = (int)(idx - (uint32_t)Ih * (uint32_t)Mh);
        const int I = 2 * Ih + (int)(q >> 1), J = 2 * Jh + (int)(q & 1u);
        // stage the patch of Fig. 3: lattice rows 4I-3 .. 4I+6, columns 4J-4 .. 4J+7
        DtilePatch P{0ull, 0ull};
#pragma unroll
        for (int pr = 0; pr < 10; ++pr) {
            const unsigned long long bits = dtile_row12<FMT>(lat, L, 4 * I - 3 + pr, 4 * J - 4);
            if (pr < 5) P.lo |= bits << (12 * pr); else P.hi |= bits << (12 * (pr - 5));
        }
        // S9: the domain and its four-neighbours lie in patch rows 2..7, columns 3..8
        constexpr unsigned long long kLoMask = (0x1F8ull << 24) | (0x1F8ull << 36) | (0x1F8ull << 48);
        constexpr unsigned long long kHiMask = 0x1F8ull | (0x1F8ull << 12) | (0x1F8ull << 24);
        const bool all0 = ((P.lo & kLoMask) | (P.hi & kHiMask)) == 0ull;
        const bool all1 = (P.lo & kLoMask) == kLoMask && (P.hi & kHiMask) == kHiMask;
        if (!all0 && !all1) {
            const unsigned long long lo0 = P.lo, hi0 = P.hi;
            const uint64_t seed = a.seeds[b];
            const uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFu), k1 = (uint32_t)(seed >> 32);
            const uint32_t d = (uint32_t)I * (uint32_t)M + (uint32_t)J, t = a.t_begin + m;
#pragma unroll 2
            for (uint32_t p = 0; p < 16u; ++p) {
                uint32_t x[4];
                philox4x32_10(d, t, p, kTagDtile, k0, k1, x);
                const int pr = 3 + (int)(x[0] >> 30), pc = 4 + (int)((x[0] >> 28) & 3u);
                const uint32_t dir = x[2] >> 30;  // 0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1)
                const int yr = pr + (dir == 0u ? -1 : dir == 1u ? 1 : 0);
                const int yc = pc + (dir == 2u ? -1 : dir == 3u ? 1 : 0);
                const int sx = P.get(pr, pc), sy = P.get(yr, yc);
                if (sx != sy) {
                    const int dA = P.A(pr, pc) - P.A(yr, yc);
                    if (x[1] < table[table_index(dA, sx - sy)]) P.toggle(pr, pc);
                }
            }
            // write the domain back (patch rows 3..6, columns 4..7) if it changed
            const unsigned long long dl = lo0 ^ P.lo, dh = hi0 ^ P.hi;
            if ((dl | dh) != 0ull) {
#pragma unroll
                for (int r4 = 0; r4 < 4; ++r4) {
                    const int pr = 3 + r4;
                    const int sh = 12 * (pr < 5 ? pr : pr - 5) + 4;
                    const uint32_t neu = (uint32_t)(((pr < 5 ? P.lo : P.hi) >> sh) & 0xFull);
                    const uint32_t chg = (uint32_t)(((pr < 5 ? dl : dh) >> sh) & 0xFull);
                    if (chg == 0u) continue;
                    const int i = 4 * I + r4;
                    if (FMT == kFmtU8) {
                        // bit n -> byte n
                        *reinterpret_cast<uint32_t*>(lat + (size_t)i * (size_t)L + 4 * J) = (neu * 0x00204081u) & 0x01010101u;
                    } else {
                        // other domains of this type share the word: flip our own bits atomically
                        atomicXor(reinterpret_cast<uint32_t*>(lat) + (size_t)i * (size_t)(L >> 5) + (size_t)(J >> 3),
                                  chg << ((4 * J) & 31));
                    }
                    delta += __popc(neu) - __popc(neu ^ chg);
                }
            }
        }
    }
    if (a.deltas != nullptr) {
        delta = __reduce_add_sync(0xFFFFFFFFu, delta);
        __shared__ int part[kDtileThreads / 32];
        if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = delta;
        __syncthreads();
        if (threadIdx.x == 0) {
            int s = 0;
            for (int w = 0; w < kDtileThreads / 32; ++w) s += part[w];
            if (s != 0)
                atomicAdd(a.deltas + (size_t)b * a.n_mcs + m, (unsigned long long)(long long)s);
        }
    }
}

inline void dtile_launch(int fmt, const PhaseArgs& a, uint32_t m, uint32_t q, uint32_t B, cudaStream_t stream)
{
    const uint32_t Mh = a.L / 8;
    dim3 grid((Mh * Mh + kDtileThreads - 1) / kDtileThreads, B);
    if (fmt == kFmtU8)
        dtile_part_kernel<kFmtU8><<<grid, kDtileThreads, 0, stream>>>(a, m, q);
    else
        dtile_part_kernel<kFmtBits><<<grid, kDtileThreads, 0, stream>>>(a, m, q);
}

}  // namespace pgg
