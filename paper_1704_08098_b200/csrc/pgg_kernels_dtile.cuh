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
// on registers only -- the 5x5 neighbourhoods of x and y are shifted to a fixed
// position, so A is two popcounts against constant masks -- flips toggle a
// register bit, and the 4x4 domain is written back once, only if it changed.
// A domain whose 6x6 neighbourhood is uniform cannot change (S9) and skips its
// 16 draws: the domains of a CTA that can change are compacted through shared
// memory first, so that warps run the pick loop with all lanes live (ncu on the
// uncompacted version: 12 of 32 lanes active on average).  Race-free in place: same-type domains are separated by 4 sites,
// reads reach 3.
// The flip count of the part is reduced per CTA into deltas[m] (a8).
#pragma once
#include <initializer_list>

#include "pgg_common.cuh"

namespace pgg {

constexpr uint32_t kTagDtile = 5u;
constexpr int kDtileThreads = 256;

struct DtilePatch {
    unsigned long long lo, hi;  // rows 0-4 / 5-9 of the patch, 12 bits each (bits 0..59 of each word)
    // The 5x5 neighbourhood of patch site (pr, pc), 2 <= pr <= 7, 2 <= pc <= 9, at fixed positions:
    // the 120-bit patch shifted right until (pr, pc) sits at bit 26 (row field 2, column 2), low 64
    // bits.  Fields 0..4 = rows pr-2 .. pr+2; columns 0..4 of a field = pc-2 .. pc+2 (the column
    // part of the shift is <= 7, so bits of the next row only reach columns >= 5 of a field).
    __device__ __forceinline__ unsigned long long window(int pr, int pc) const
    {
        const int s = 12 * (pr - 2) + (pc - 2);  // 0 .. 67
        return s < 60 ? (lo >> s) | (hi << (60 - s)) : hi >> (s - 60);
    }
    __device__ __forceinline__ void toggle(int pr, int pc)
    {
        const unsigned long long bit = 1ull << (12 * (pr < 5 ? pr : pr - 5) + pc);
        if (pr < 5) lo ^= bit; else hi ^= bit;
    }
};

// s and A of the site at the centre (bit 26) of a window: A = 5 s + 2 (nearest + diagonal) +
// axial distance-2 (include/pgg.h); one row = 12 bits
constexpr int kDtileCentre = 26;
constexpr unsigned long long dtile_bits(std::initializer_list<int> offs)
{
    unsigned long long m = 0;
    for (int o : offs) m |= 1ull << (kDtileCentre + o);
    return m;
}
constexpr unsigned long long kDtileW2 = dtile_bits({-1, 1, -12, 12, -13, -11, 11, 13});
constexpr unsigned long long kDtileW1 = dtile_bits({-2, 2, -24, 24});
__device__ __forceinline__ int dtile_s(unsigned long long w) { return (int)((w >> kDtileCentre) & 1ull); }
// 2 (nearest + diagonal) + axial distance-2 of the centre site, i.e. A - 5 s.  The weight-2 bits span
// 27 positions (centre -13 .. +13) and the weight-1 bits fold into one word without colliding (bits
// 2, 24, 28 and 50 - 32 = 18), so each sum is ONE 32-bit population count (POPC issues at a fraction
// of the ALU rate).
__device__ __forceinline__ int dtile_nbsum(unsigned long long w)
{
    static_assert(kDtileCentre == 26, "the folding below assumes the centre at bit 26");
    const uint32_t w2 = (uint32_t)(w >> 13) & (uint32_t)(kDtileW2 >> 13);
    const unsigned long long a = w & kDtileW1;
    const uint32_t w1 = (uint32_t)a | (uint32_t)(a >> 32);
    return 2 * __popc(w2) + __popc(w1);
}

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
    // domains that can change, compacted over the CTA: (patch, I << 16 | J)
    __shared__ unsigned long long s_lo[kDtileThreads], s_hi[kDtileThreads];
    __shared__ uint32_t s_ij[kDtileThreads];
    __shared__ uint32_t s_n;
    const uint32_t b = blockIdx.y;
    const int L = (int)a.L, M = L >> 2, Mh = M >> 1;
    uint8_t* lat = a.lats + (size_t)b * a.lat_bytes;
    const uint32_t* __restrict__ table = a.tables + (size_t)b * kTableSize;
    const uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    if (threadIdx.x == 0) s_n = 0u;
    __syncthreads();
    {
        DtilePatch P{0ull, 0ull};
        int I = 0, J = 0;
        bool active = false;
        if (idx < (uint32_t)Mh * (uint32_t)Mh) {
            const int Ih = (int)(idx / (uint32_t)Mh), Jh = (int)(idx - (uint32_t)Ih * (uint32_t)Mh);
            I = 2 * Ih + (int)(q >> 1);
            J = 2 * Jh + (int)(q & 1u);
            // stage the patch of Fig. 3: lattice rows 4I-3 .. 4I+6, columns 4J-4 .. 4J+7
#pragma unroll
            for (int pr = 0; pr < 10; ++pr) {
                const unsigned long long bits = dtile_row12<FMT>(lat, L, 4 * I - 3 + pr, 4 * J - 4);
                if (pr < 5) P.lo |= bits << (12 * pr); else P.hi |= bits << (12 * (pr - 5));
            }
            // S9: the domain and its four-neighbours lie in patch rows 2..7, columns 3..8; if they
            // all hold one strategy no pick can change the domain and its 16 draws are skipped
            constexpr unsigned long long kLoMask = (0x1F8ull << 24) | (0x1F8ull << 36) | (0x1F8ull << 48);
            constexpr unsigned long long kHiMask = 0x1F8ull | (0x1F8ull << 12) | (0x1F8ull << 24);
            const bool all0 = ((P.lo & kLoMask) | (P.hi & kHiMask)) == 0ull;
            const bool all1 = (P.lo & kLoMask) == kLoMask && (P.hi & kHiMask) == kHiMask;
            active = !all0 && !all1;
        }
        const uint32_t mk = __ballot_sync(0xFFFFFFFFu, active);
        uint32_t base = 0;
        if (lane == 0 && mk != 0u) base = atomicAdd(&s_n, (uint32_t)__popc(mk));
        base = __shfl_sync(0xFFFFFFFFu, base, 0);
        if (active) {
            const uint32_t pos = base + (uint32_t)__popc(mk & ((1u << lane) - 1u));
            s_lo[pos] = P.lo;
            s_hi[pos] = P.hi;
            s_ij[pos] = ((uint32_t)I << 16) | (uint32_t)J;
        }
    }
    __syncthreads();
    int delta = 0;
    if (threadIdx.x < s_n) {
        DtilePatch P{s_lo[threadIdx.x], s_hi[threadIdx.x]};
        const int I = (int)(s_ij[threadIdx.x] >> 16), J = (int)(s_ij[threadIdx.x] & 0xFFFFu);
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
            const unsigned long long wx = P.window(pr, pc), wy = P.window(yr, yc);
            const int sx = dtile_s(wx), sy = dtile_s(wy);
            // branch-free: with 32 live domains per warp some lane nearly always needs the payoffs
            const int dA = 5 * (sx - sy) + dtile_nbsum(wx) - dtile_nbsum(wy);
            const uint32_t T = table[table_index(dA, sx - sy)];
            if (sx != sy && x[1] < T) P.toggle(pr, pc);
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
