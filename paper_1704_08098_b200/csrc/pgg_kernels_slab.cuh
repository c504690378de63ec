// pgg_kernels_slab.cuh -- one phase on a ROW SLAB of a lattice that is sharded over several GPUs
// ("1-D row slabs, after each phase exchange the 3 boundary rows each way ...
// fuse the halo push into the phase kernel"; the periodic L x L lattice is PAPER.md:45).
//
// A slab is lattice rows [row0, row0 + n_rows) plus three halo rows on either side (the read stencil of
// an elementary step has radius 3): buffer row q holds lattice row (row0 - 3 + q) mod L,
// q = 0 .. n_rows + 5, whole rows, in the canonical layout of the lattice (uint8 or bit-packed).
// Columns stay periodic inside the slab; rows never wrap (the halo rows are the periodic images).
//
// The step is V0's (uint8: one thread per active site of the slab's own rows; bit-packed: one thread per
// 32-site word, the S9 scan of eight sites in ten logic operations; plain global loads) with the site index
// of the GLOBAL lattice in the Philox counter, so every slab draws exactly what the unsharded sweep draws:
// the result is bit-identical to pgg_sweep whatever the number of slabs.
//
// Halo push, fused.  A site of the slab's first (last) three own rows is also a halo site of the upper
// (lower) neighbour slab.  The thread that flips it stores the new value into the neighbour's halo copy as
// well, through `up_halo` / `dn_halo` -- plain device pointers, local or peer (NVLink P2P) memory.  Within
// a phase nobody reads those copies: a step reads no site of the active class but its own x (same-class
// sites are >= 4 apart), so the push races with nothing; BETWEEN phases the slabs must be ordered.
//
// Ordering between phases, without the host.  flags[1] / flags[2] of a slab count the phases its upper /
// lower neighbour has completed (written by that neighbour, release at system scope); a phase with global
// number `epoch` starts when both are >= epoch (so the neighbours' pushes of all earlier phases have
// landed AND the neighbours have finished reading what this phase is about to overwrite ... one phase of
// skew at most), and the last CTA to finish posts epoch + 1 to both neighbours.  flags[0] is the CTA
// counter of that "last one out" detection.  With flags == nullptr the caller orders the phases itself
// (slabs of one device on one stream: the test path).
#pragma once
#include "pgg_common.cuh"

namespace pgg {

struct SlabArgs {
    uint8_t* slab;               // (n_rows + 6) rows
    uint8_t* up_halo;            // three rows: the copy of this slab's own rows 0..2 held by the upper neighbour
    uint8_t* dn_halo;            // three rows: the copy of own rows n_rows-3 .. n_rows-1 held by the lower neighbour
    const uint64_t* seed;
    const uint32_t* table;       // 153 thresholds
    const uint8_t* order;        // [n_mcs spanned][16] phase classes, row 0 = MCS t0
    unsigned long long* deltas;  // [n_mcs spanned] signed flip sums of this slab's rows, ACCUMULATED; or nullptr
    unsigned int* flags;         // this slab's three words (see above) or nullptr
    unsigned int* up_flag;       // the upper neighbour's flags[2] (this slab is its lower neighbour)
    unsigned int* dn_flag;       // the lower neighbour's flags[1]
    uint32_t L, row0, n_rows;
    uint32_t t0;                 // MCS of order[0] / deltas[0]
};

// Buffer-row accessor with the get(i, j) interface payoff_A / pd_neighbour_count expect: i is a BUFFER row
// (never wrapped), j a column in [-4, L + 4).
template <int FMT>
struct SlabLattice;

template <>
struct SlabLattice<kFmtU8> {
    uint8_t* p;
    int L;
    __device__ __forceinline__ int get(int q, int j) const { return p[(size_t)q * (size_t)L + (size_t)wrap_coord(j, L)]; }
    static __device__ __forceinline__ void set(uint8_t* rows, int L, int q, int j, int v)
    {
        rows[(size_t)q * (size_t)L + (size_t)j] = (uint8_t)v;
    }
};

template <>
struct SlabLattice<kFmtBits> {
    uint8_t* p;
    int L;
    __device__ __forceinline__ int get(int q, int j) const
    {
        const int jj = wrap_coord(j, L);
        const uint32_t w = reinterpret_cast<const uint32_t*>(p)[(size_t)q * (size_t)(L >> 5) + (size_t)(jj >> 5)];
        return (int)((w >> (jj & 31)) & 1u);
    }
    // eight sites of a class share a word: set / clear the bit atomically (idempotent, unlike a flip)
    static __device__ __forceinline__ void set(uint8_t* rows, int L, int q, int j, int v)
    {
        uint32_t* w = reinterpret_cast<uint32_t*>(rows) + (size_t)q * (size_t)(L >> 5) + (size_t)(j >> 5);
        if (v) atomicOr(w, 1u << (j & 31)); else atomicAnd(w, ~(1u << (j & 31)));
    }
};

// The start of a phase: wait until both neighbours have completed `epoch` phases.
__device__ __forceinline__ void slab_wait(const SlabArgs& a, uint32_t epoch)
{
    if (a.flags == nullptr) return;
    if (threadIdx.x == 0) {
        unsigned int s1, s2, spins = 0;
        for (;;) {
            asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(s1) : "l"(a.flags + 1) : "memory");
            asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(s2) : "l"(a.flags + 2) : "memory");
            if (s1 >= epoch && s2 >= epoch) break;
            __nanosleep(200);
            if (++spins > (1u << 23)) __trap();  // seconds: a lost neighbour must not hang the device
        }
    }
    __syncthreads();
}

// Kernels whose CTAs own contiguous row bands (LEAN on a slab) need less: only the FIRST band reads the top halo
// and pushes upwards, only the LAST band reads the bottom halo and pushes downwards, and the bands of one slab are
// ordered among themselves by the launches.  So only those two CTAs wait (each for its own neighbour) and post
// (each to its own neighbour): no ticket counter, no last-one-out chain; flags[0] is not used.
__device__ __forceinline__ void slab_wait_edge(const SlabArgs& a, uint32_t epoch, bool top, bool bottom)
{
    if (a.flags == nullptr || !(top || bottom)) return;
    if (threadIdx.x == 0) {
        unsigned int s1 = epoch, s2 = epoch, spins = 0;
        for (;;) {
            if (top) asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(s1) : "l"(a.flags + 1) : "memory");
            if (bottom) asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(s2) : "l"(a.flags + 2) : "memory");
            if (s1 >= epoch && s2 >= epoch) break;
            __nanosleep(200);
            if (++spins > (1u << 23)) __trap();
        }
    }
    __syncthreads();
}

// thread 0, after a __syncthreads that follows every store of the CTA
__device__ __forceinline__ void slab_post_edge(const SlabArgs& a, uint32_t epoch, bool top, bool bottom)
{
    if (a.flags == nullptr || !(top || bottom)) return;
    __threadfence_system();  // fence + relaxed store = release: the band's flips and pushes before its flag
    const unsigned int next = epoch + 1u;
    if (top) asm volatile("st.relaxed.sys.global.u32 [%0], %1;" ::"l"(a.up_flag), "r"(next) : "memory");
    if (bottom) asm volatile("st.relaxed.sys.global.u32 [%0], %1;" ::"l"(a.dn_flag), "r"(next) : "memory");
}

// The end of a phase, thread 0 of a CTA whose stores are all ordered before this call (after a __syncthreads):
// its ticket, and -- by the last CTA out -- epoch + 1 to both neighbours.
__device__ __forceinline__ void slab_post(const SlabArgs& a, uint32_t epoch)
{
    if (a.flags == nullptr) return;
    __threadfence_system();  // this CTA's stores (own rows, pushes into the neighbours) before its ticket
    const unsigned int done = atomicAdd(a.flags, 1u);
    if (done == gridDim.x - 1u) {  // last CTA out
        atomicExch(a.flags, 0u);
        // fence - ticket ... ticket - fence: every CTA's stores are ordered before what follows, system-wide;
        // fence + relaxed store = the release of epoch + 1 to the neighbours
        __threadfence_system();
        const unsigned int next = epoch + 1u;
        asm volatile("st.relaxed.sys.global.u32 [%0], %1;" ::"l"(a.up_flag), "r"(next) : "memory");
        asm volatile("st.relaxed.sys.global.u32 [%0], %1;" ::"l"(a.dn_flag), "r"(next) : "memory");
    }
}

// The end of a phase for the kernels of this file: the CTA's flip count, then slab_post.
__device__ __forceinline__ void slab_finish(const SlabArgs& a, int delta, uint32_t t, uint32_t epoch)
{
    __shared__ int part[8];
    delta = __reduce_add_sync(0xFFFFFFFFu, delta);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = delta;
    __syncthreads();  // also: every store of this CTA (own rows, halo pushes) is ordered before thread 0's fence
    if (threadIdx.x == 0) {
        int s = 0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += part[w];
        if (s != 0 && a.deltas != nullptr) atomicAdd(a.deltas + (t - a.t0), (unsigned long long)(long long)s);
        slab_post(a, epoch);
    }
}

// a5-a7 for a site x = (buffer row q, column j) whose drawn neighbour differs: payoff difference (public goods game)
// or the neighbour counts of x and y (prisoner's dilemma; nx = cooperators among x's four neighbours),
// threshold compare, write with the halo push.  Returns the change of the cooperator count.
template <int FMT, int GAME>
__device__ __forceinline__ int slab_accept(const SlabArgs& a, const SlabLattice<FMT>& lat, int q, int j, int dir, int sx,
                                           int sy, int nx, uint32_t u)
{
    const int L = lat.L, n_rows = (int)a.n_rows, own = q - 3;
    const int yq = q + (dir == 0 ? -1 : dir == 1 ? 1 : 0);
    const int yj = j + (dir == 2 ? -1 : dir == 3 ? 1 : 0);
    const int idx_t = GAME == kGamePD ? sx * 25 + nx * 5 + pd_neighbour_count(lat, yq, yj)
                                      : table_index(payoff_A(lat, q, j) - payoff_A(lat, yq, yj), sx - sy);
    if (u >= a.table[idx_t]) return 0;
    SlabLattice<FMT>::set(a.slab, L, q, j, sy);
    if (own < 3) SlabLattice<FMT>::set(a.up_halo, L, own, j, sy);
    if (own >= n_rows - 3) SlabLattice<FMT>::set(a.dn_halo, L, own - (n_rows - 3), j, sy);
    return sy - sx;
}

// uint8 slabs: one thread per active site (V0's step).  A fixed grid strides over the sites, so the flag
// protocol costs one wait and one post per CTA whatever the slab's size.
template <int FMT, int GAME = kGamePGG>
__global__ void __launch_bounds__(256)
phase_slab_kernel(SlabArgs a, uint32_t t, uint32_t k, uint32_t epoch)
{
    slab_wait(a, epoch);
    const uint32_t cls = a.order[(size_t)(t - a.t0) * 16 + k];
    const int ci = (int)(cls >> 2), cj = (int)(cls & 3u);
    const StepKey sk = make_step_key(a.seed[0], t, k, cls);
    const int L = (int)a.L, m4 = L >> 2;
    SlabLattice<FMT> lat{a.slab, L};
    const uint32_t n_cls = (a.n_rows >> 2) * (uint32_t)m4;
    int delta = 0;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n_cls; idx += gridDim.x * blockDim.x) {
        const int bi = (int)(idx / (uint32_t)m4), bj = (int)(idx - (uint32_t)bi * (uint32_t)m4);
        const int own = 4 * bi + ci;        // own row of the slab, 0 .. n_rows - 1
        const int q = own + 3, j = 4 * bj + cj;
        const uint32_t gi = a.row0 + (uint32_t)own;  // lattice row (row0 + n_rows <= L: never wraps)
        const int sx = lat.get(q, j);
        const int s_up = lat.get(q - 1, j), s_dn = lat.get(q + 1, j);
        const int s_lf = lat.get(q, j - 1), s_rt = lat.get(q, j + 1);
        const int nx = s_up + s_dn + s_lf + s_rt;
        if (nx != 4 * sx) {  // S9
            uint32_t x0, u;
            step_draw(sk, gi * (uint32_t)L + (uint32_t)j, x0, u);
            const int dir = (int)(x0 >> 30);  // 0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1)
            const int sy = dir == 0 ? s_up : dir == 1 ? s_dn : dir == 2 ? s_lf : s_rt;
            if (sy != sx) delta += slab_accept<FMT, GAME>(a, lat, q, j, dir, sx, sy, nx, u);
        }
    }
    slab_finish(a, delta, t, epoch);
}

// Bit-packed slabs: one thread per 32-site word of an active row -- eight active sites.  Five coalesced word
// loads and ten logic operations say which of the eight have a neighbour of the other strategy (S9; the
// scan of the LEAN kernel, on global memory); the thread then walks those sites.  Later sites of the word
// see nothing of the earlier ones' flips: they are of the same class, and a step reads no site of the
// active class but its own.
template <int GAME = kGamePGG>
__global__ void __launch_bounds__(256)
phase_slab_words_kernel(SlabArgs a, uint32_t t, uint32_t k, uint32_t epoch)
{
    slab_wait(a, epoch);
    const uint32_t cls = a.order[(size_t)(t - a.t0) * 16 + k];
    const int ci = (int)(cls >> 2), cj = (int)(cls & 3u);
    const StepKey sk = make_step_key(a.seed[0], t, k, cls);
    const int L = (int)a.L, W = L >> 5;
    SlabLattice<kFmtBits> lat{a.slab, L};
    const uint32_t* words = reinterpret_cast<const uint32_t*>(a.slab);
    const uint32_t n_words = (a.n_rows >> 2) * (uint32_t)W;
    const uint32_t cm = 0x11111111u << cj;  // the active sites of a word
    int delta = 0;
    for (uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x; idx < n_words; idx += gridDim.x * blockDim.x) {
        const int bi = (int)(idx / (uint32_t)W), kw = (int)(idx - (uint32_t)bi * (uint32_t)W);
        const int own = 4 * bi + ci, q = own + 3;
        const uint32_t* row = words + (size_t)q * (size_t)W;
        const uint32_t c = row[kw], up = row[kw - W], dn = row[kw + W];
        const uint32_t pv = row[kw == 0 ? W - 1 : kw - 1], nx = row[kw == W - 1 ? 0 : kw + 1];
        const uint32_t lf = __funnelshift_l(pv, c, 1), rt = __funnelshift_r(c, nx, 1);  // bit p = site p - 1 / p + 1
        uint32_t nb = ((c ^ up) | (c ^ dn) | (c ^ lf) | (c ^ rt)) & cm;
        const uint32_t site0 = (a.row0 + (uint32_t)own) * (uint32_t)L + 32u * (uint32_t)kw;
        while (nb) {
            const int p = __ffs((int)nb) - 1;
            nb &= nb - 1u;
            uint32_t x0, u;
            step_draw(sk, site0 + (uint32_t)p, x0, u);
            const int dir = (int)(x0 >> 30);
            const uint32_t ny = dir == 0 ? up : dir == 1 ? dn : dir == 2 ? lf : rt;
            const int sx = (int)((c >> p) & 1u), sy = (int)((ny >> p) & 1u);
            const int n4 = (int)(((up >> p) & 1u) + ((dn >> p) & 1u) + ((lf >> p) & 1u) + ((rt >> p) & 1u));
            if (sy != sx) delta += slab_accept<kFmtBits, GAME>(a, lat, q, 32 * kw + p, dir, sx, sy, n4, u);
        }
    }
    slab_finish(a, delta, t, epoch);
}

}  // namespace pgg
