// pgg_kernels_lean.cuh -- the LEAN phase kernel (K1 uint8, K2 bit-packed): whatever the
// layout in HBM, the on-chip copy of the lattice is BIT-PACKED.
//
// Why (round-2 measurements, profiles/r2_*): RING (uint8) and BAND (bit-packed) both execute
// ~41 M warp instructions per L = 16384 phase -- 2.4 per active site -- and are bound by
// instruction issue at 58-64 % with one 17-warp CTA per SM.  RING spends 37 % of them scanning
// bytes (one active byte per 32-bit word), and its 32 KB uint8 ring slots stay live for three
// steps, so half of the 227 KB ring never prefetches.  A Philox-only kernel draws 5.2e11 sites/s
// (pgg_probe_draw_rate), i.e. the draws of a phase need ~9 us; the rest was overhead.
//
//   * full lattice rows stream through shared memory (a band of consecutive rows per
//     persistent CTA; rows are contiguous in global memory, so a staging slot of up to 32 KB
//     arrives as ONE cp.async.bulk, SASS UBLKCP, completing on an mbarrier);
//   * uint8 source: the 16 consumer warps PACK each staged row to bits on arrival
//     (16 bytes -> 16 bits with four multiplies: bytes b0..b3 of a word times 0x00204081 put
//     b0 b1 b2 b3 at bits 21..24) into a small ring of bit rows and hand the staging slot
//     straight back to the producer -- every uint8 slot prefetches, none is "live";
//   * bit-packed source: the rows land in the bit ring directly;
//   * the bit ring holds 6+ chunks (L = 16384: 2 KB per row), with the last three rows
//     mirrored in front of row 0, so no stencil read ever wraps;
//   * scan (a4, S9): one 32-site word per lane and step -- eight active sites -- with five
//     shared loads and ten logic operations;
//   * survivors are extracted lane-serially after a warp prefix sum (one FLO + one 8-byte
//     store per survivor) into the warp's queue Q1 = (ring bit offset, site);
//   * level 1 (a3, a4): Philox on dense batches of 32 (two batches interleaved when 64 wait);
//     sites whose drawn neighbour differs go to Q2 with their u;
//   * level 2 (a5-a7): the 14-read signed stencil on dense batches of 32, threshold compare,
//     in-place write to the lattice in HBM (byte store / atomicXor), flip count (a8).
//
// Geometry.  n_groups = L/4 active rows per class.  A step = R active rows (R*L/32 = 512 words,
// one per lane of the 16 consumer warps; rows longer than 16384 sites take n_seg segments).
// chunk c = RC = 4R consecutive lattice rows starting at an active row; step s reads the tail
// of chunk s and chunk s+1.  Band = steps [S0, S1) of one lattice for one CTA.
//
// Queue lifetime.  A queued site is finished within `lag` steps: both queues are drained at the
// end of every lag-th step (and of the band), in between only full batches of 32 run.  (RING had
// to finish a site within one step because its 32 KB uint8 slots were too dear to keep; there Q2
// filled its batches only half.)  The bit ring keeps the rows that long: lag + 3 chunks or more.
//
// Roles.  Warp 16 issues the bulk copies.  uint8 source: four PACKER warps (17..20) wait for a
// staging slot, pack their share of it into the ring chunk, hand the slot back (stage empty) and,
// when a chunk is complete, arrive on the chunk's "full" barrier; they wait for the chunk's
// "empty" barrier before they overwrite it.  The 16 WORKER warps (0..15) see the same protocol
// for both sources -- full/empty mbarriers per ring chunk, "full" completed by the bulk copy
// (bit-packed) or by the packers (uint8); chunk s-lag is released at the end of step s (every site
// that reads it was queued in a step <= s-lag and has been drained by then).  Packing is a steady
// stream beside the workers instead of a burst in front of every step, so the staging slots
// refill continuously, and the SM holds 21 warps instead of 17.
#pragma once
#include "pgg_kernels_ring.cuh"
#include "pgg_stencil_lut.cuh"
#include "pgg_kernels_slab.cuh"

namespace pgg {

constexpr int kLeanConsumers = 16;
constexpr int kLeanPackers = 4;   // uint8 source: warps that turn staged bytes into ring bits
constexpr int kLeanThreads = (kLeanConsumers + 1) * 32;                    // bit-packed source
constexpr int kLeanThreadsU8 = (kLeanConsumers + 1 + kLeanPackers) * 32;   // uint8 source
constexpr int kLeanQ1Cap = 192;   // 8-byte entries per warp: leftover (< 64) + at most 128 per extraction round
constexpr int kLeanQ2Cap = 64;    // 16-byte entries per warp (a ring: power of two)
constexpr int kLeanWarpQBytes = kLeanQ1Cap * 8 + kLeanQ2Cap * 16;
constexpr int kLeanMaxSlots = 12; // staging slots (uint8) / ring chunks (bit-packed): barrier array size
constexpr int kLeanLagU8 = 4;     // ring chunks >= lag + 3 (see "Queue lifetime"); the rest runs ahead
constexpr int kLeanLagBits = 8;
constexpr int kLeanFixedBytes = kLeanConsumers * kLeanWarpQBytes + 160 * 4 + 4 * kLeanMaxSlots * 8 + 8 * 4 + kStencilLutBytes + 128;

struct LeanPlan {
    uint32_t lg2L;       // L = 2^lg2L sites per row = bits per ring row
    uint32_t pitch;      // bytes per ring row = L / 8
    uint32_t lgWPR;      // log2(words per row)
    uint32_t R;          // active rows per step
    uint32_t RC;         // lattice rows per chunk = 4 R
    uint32_t n_seg;      // segments of 512 words per active row (L > 16384), else 1
    uint32_t NR;         // chunks in the bit ring
    uint32_t lag;        // a queued site is finished within `lag` steps (power of two)
    uint32_t SR;         // uint8: rows per staging slot
    uint32_t SPC;        // uint8: staging slots per chunk = RC / SR
    uint32_t NS;         // uint8: staging slots
    uint32_t slot_bytes; // uint8: SR * L
    uint32_t nb;         // bands (CTAs) per lattice
    uint32_t n_steps_total;  // (L / 4) / R; a row slab: (n_rows / 4) / R
    uint32_t smem_bytes;
    uint32_t step0;      // a row slab (SLAB): its first step = (row0 / 4) / R; else 0
};

// 16 lattice bytes (0 / 1 each) -> 16 bits (bit s = byte s) in the low half; the high half is junk.
__device__ __forceinline__ uint32_t lean_pack16(uint4 v)
{
    constexpr uint32_t M = 0x00204081u;  // 2^21 + 2^14 + 2^7 + 1: no two partial products meet, so no carries
    const uint32_t p0 = v.x * M, p1 = v.y * (M << 4);  // bytes of v.x at bits 21..24, of v.y at 25..28
    const uint32_t p2 = v.z * M, p3 = v.w * (M << 4);
    constexpr uint32_t m = 0x01E00000u;
    const uint32_t lo = (p0 & m) | (p1 & ~m);          // bits 21..28 = sites 0..7 (one LOP3)
    const uint32_t hi = (p2 & m) | (p3 & ~m);          // bits 21..28 = sites 8..15
    const uint32_t a = lo >> 21, b2 = hi >> 13;
    return (a & 0xFFu) | (b2 & ~0xFFu);                // bits 0..7 | bits 8..15 (| junk above)
}

// Ballot of bit `BIT` of v over the full warp.  (and + setp.ne in PTX become one LOP3 that writes the predicate;
// the C++ form compiled to a shift, an and and a compare per ballot.)
template <int BIT>
__device__ __forceinline__ uint32_t ballot_bit(uint32_t v)
{
    uint32_t r;
    asm volatile(
        "{\n\t.reg .pred p;\n\t.reg .b32 t;\n\t"
        "and.b32 t, %1, %2;\n\t"
        "setp.ne.u32 p, t, 0;\n\t"
        "vote.sync.ballot.b32 %0, p, 0xffffffff;\n\t}"
        : "=r"(r)
        : "r"(v), "n"(1u << BIT));
    return r;
}

// The producer's wait: it has a whole step of slack, so it backs off instead of competing for issue slots.
__device__ __forceinline__ void mbar_wait_relaxed(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    for (;;) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
        if (done) break;
        __nanosleep(100);
    }
}

__device__ __forceinline__ void mbar_arrive_cta(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// SRC = layout of the lattice in global memory (kFmtU8 / kFmtBits); the ring is always bits.
// Warps 0..15: workers.  Warp 16: producer (bulk copies).  Warps 17..20 (uint8 only): packers.
// GAME = kGamePGG (the 14-read payoff stencil) or kGamePD (neighbour counts of x and y).
// PERSIST: called once per phase from the persistent kernel (no programmatic-dependent-launch fences;
// the mbarriers are initialised afresh, which is legal because every warp has passed the closing
// __syncthreads of the previous phase).
// SLAB: the "lattice" is a row slab of a lattice sharded over several GPUs
// (pgg_kernels_slab.cuh).  a.lats is the VIRTUAL base -- the address lattice row 0 would have, so that lattice
// row i of the slab's buffer (own rows and halo rows) is at a.lats + i * (bytes per row), i = row0 - 3 .. row0 + n_rows + 2,
// possibly negative or >= L: rows never wrap, the halo rows are the periodic images.  The steps are those of the
// whole lattice (g.step0 = the slab's first), so sites and draws are the unsharded sweep's.  A flip in the first /
// last three own rows is pushed into the neighbour's halo copy; the phase starts when both neighbours have
// completed `epoch` phases; only the first and the last band wait and post (slab_wait_edge / slab_post_edge).
template <int SRC, int GAME, bool PERSIST, bool SLAB = false>
__device__ __forceinline__ void lean_phase(const PhaseArgs& a, uint32_t m, uint32_t k, const LeanPlan& g, bool tables = true,
                                           const SlabArgs* sl = nullptr, uint32_t epoch = 0)
{
    static_assert(!SLAB || !PERSIST, "row slabs: one launch per phase");
    extern __shared__ __align__(128) uint8_t smem_raw[];
    const int pitch = (int)g.pitch, RC = (int)g.RC;
    const uint32_t NR = g.NR;
    const int chunk_bytes = RC * pitch;
    const int ring_bytes = (int)NR * chunk_bytes;
    const int ring_off = 3 * pitch;                         // three mirror rows in front of ring row 0
    uint8_t* ring0 = smem_raw + ring_off;
    const int stage_off = ring_off + ring_bytes;            // uint8 source only
    const int q_off = stage_off + (SRC == kFmtU8 ? (int)(g.NS * g.slot_bytes) : 0);
    uint32_t* tbl = reinterpret_cast<uint32_t*>(smem_raw + q_off + kLeanConsumers * kLeanWarpQBytes);
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(tbl + 160);  // ring full[], ring empty[], stage full[], stage empty[]
    int* eoff = reinterpret_cast<int*>(bars + 4 * kLeanMaxSlots);                 // e[4], f[4]
    int8_t* lut = reinterpret_cast<int8_t*>(eoff + 8);                            // StencilLut
    __shared__ int delta_cta;

    const uint32_t b = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t L = a.L;
    uint8_t* lat = a.lats + (size_t)b * a.lat_bytes;
    const uint32_t bar_full = smem_u32(bars), bar_empty = bar_full + 8u * kLeanMaxSlots;   // of the bit ring's chunks
    const uint32_t bar_sfull = bar_empty + 8u * kLeanMaxSlots, bar_sempty = bar_sfull + 8u * kLeanMaxSlots;  // of the staging slots

    if (!PERSIST) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (tables) {  // (PERSIST: shared memory keeps them from phase to phase)
        for (int q = threadIdx.x; q < kTableSize; q += blockDim.x)
            tbl[q] = a.tables[(size_t)b * kTableSize + q];
        if (GAME == kGamePGG)
            for (int q = threadIdx.x; q < kStencilLutBytes / 4; q += blockDim.x)
                reinterpret_cast<uint32_t*>(lut)[q] = reinterpret_cast<const uint32_t*>(g_stencil_lut.v)[q];
    }
    if (threadIdx.x == 0) {
        delta_cta = 0;
        for (uint32_t s = 0; s < NR; ++s) {
            mbar_init(bar_full + 8u * s, SRC == kFmtU8 ? kLeanPackers : 1);  // packers arrive / the bulk copy completes
            mbar_init(bar_empty + 8u * s, kLeanConsumers);
        }
        if (SRC == kFmtU8)
            for (uint32_t s = 0; s < g.NS; ++s) {
                mbar_init(bar_sfull + 8u * s, 1);
                mbar_init(bar_sempty + 8u * s, kLeanPackers);
            }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        const int ps = (int)L;  // one ring row down, in bits
        eoff[0] = -ps; eoff[1] = ps; eoff[2] = -1; eoff[3] = 1;
        eoff[4] = 1;   eoff[5] = 1;  eoff[6] = ps; eoff[7] = ps;
    }
    __syncthreads();
    // the first / last band waits until the upper / lower neighbour slab has completed the previous phase (its pushes
    // are in my halo rows, its reads of its own halo copy are over); the other bands touch no halo row.  In front of
    // griddepcontrol.wait: the flags are the neighbours' business, not the previous launch's, so the acquire's
    // latency overlaps the tail of this slab's previous phase
    if (SLAB) slab_wait_edge(*sl, epoch, blockIdx.x == 0, blockIdx.x == gridDim.x - 1);
    if (!PERSIST) asm volatile("griddepcontrol.wait;" ::: "memory");
    const uint32_t cls = a.order[((size_t)b * a.order_stride + (m % a.order_stride)) * 16 + k];
    const int ci = (int)(cls >> 2), cj = (int)(cls & 3u);

    const uint32_t band = blockIdx.x;
    const uint32_t S0 = (SLAB ? g.step0 : 0u) + (uint32_t)(((unsigned long long)band * g.n_steps_total) / g.nb);
    const uint32_t S1 = (SLAB ? g.step0 : 0u) + (uint32_t)(((unsigned long long)(band + 1) * g.n_steps_total) / g.nb);
    const uint32_t n_steps = S1 - S0;
    const uint32_t n_chunks = n_steps ? n_steps + 1 : 0;
    // first lattice row of chunk 0 (the chunk in front of the band's first active row); may be < 0
    const int row_c0 = 4 * (int)(S0 * g.R) + ci - RC;
    const uint32_t row_bytes_g = SRC == kFmtU8 ? L : L >> 3;  // bytes per lattice row in global memory

    if (warp == kLeanConsumers) {
        // ---------------- producer warp ----------------
        // PERSIST: the flips of the previous phase were made by other SMs through the generic proxy; the
        // grid barrier has ordered them before this point, this fence orders them before the bulk copies
        // SLAB: likewise for what the neighbours pushed into my halo rows (ordered before here by the flags)
        if (PERSIST || SLAB) asm volatile("fence.proxy.async.global;" ::: "memory");
        int grow = (!SLAB && row_c0 < 0) ? row_c0 + (int)L : row_c0;  // lattice row of the current chunk's first row
        if (SRC == kFmtU8) {
            const uint32_t stage_s = smem_u32(smem_raw + stage_off);
            uint32_t slot = 0, par = 0;  // wait parity of "empty": (use - 1) & 1, use = earlier fills of this slot (>= 1 after the first lap)
            bool first_lap = true;
            for (uint32_t c = 0; c < n_chunks; ++c) {
                for (uint32_t j = 0; j < g.SPC; ++j) {
                    int r0 = (int)(j * g.SR);
                    const int r1 = r0 + (int)g.SR;
                    if (c == 0) {  // of the chunk in front of the band only the last three rows are read
                        if (r1 <= RC - 3) continue;
                        r0 = max(r0, RC - 3);
                    }
                    if (!first_lap) mbar_wait_relaxed(bar_sempty + 8u * slot, par);
                    if (lane == 0) {
                        const uint32_t bar = bar_sfull + 8u * slot;
                        const int n = r1 - r0;
                        mbar_expect_tx(bar, (uint32_t)n * L);
                        int g0 = grow + r0;
                        if (!SLAB && g0 >= (int)L) g0 -= (int)L;
                        const int n1st = SLAB ? n : min(n, (int)L - g0);
                        const uint32_t dst = stage_s + slot * g.slot_bytes + (uint32_t)(r0 - (int)(j * g.SR)) * L;
                        bulk_g2s(dst, lat + (ptrdiff_t)g0 * (ptrdiff_t)L, (uint32_t)n1st * L, bar);
                        if (n1st < n) bulk_g2s(dst + (uint32_t)n1st * L, lat, (uint32_t)(n - n1st) * L, bar);
                    }
                    __syncwarp();
                    if (++slot == g.NS) { slot = 0; if (first_lap) first_lap = false; else par ^= 1u; }
                }
                grow += RC;
                if (!SLAB && grow >= (int)L) grow -= (int)L;
            }
        } else {
            const uint32_t ring_s = smem_u32(ring0);
            uint32_t slot = 0, par = 0;
            bool first_lap = true;
            for (uint32_t c = 0; c < n_chunks; ++c) {
                if (!first_lap) mbar_wait_relaxed(bar_empty + 8u * slot, par);
                if (lane == 0) {
                    const uint32_t bar = bar_full + 8u * slot;
                    const int r0 = c == 0 ? RC - 3 : 0;
                    const int n = RC - r0;
                    const bool mirror = slot == NR - 1;  // its last three rows are also staged in front of row 0
                    mbar_expect_tx(bar, (uint32_t)(n + (mirror ? 3 : 0)) * row_bytes_g);
                    int g0 = grow + r0;
                    if (!SLAB && g0 >= (int)L) g0 -= (int)L;
                    const int n1st = SLAB ? n : min(n, (int)L - g0);  // (a slab's rows never wrap; g0 may be < 0 or >= L)
                    const uint32_t dst = ring_s + (slot * (uint32_t)RC + (uint32_t)r0) * (uint32_t)pitch;
                    bulk_g2s(dst, lat + (ptrdiff_t)g0 * (ptrdiff_t)row_bytes_g, (uint32_t)n1st * row_bytes_g, bar);
                    if (n1st < n) bulk_g2s(dst + (uint32_t)n1st * row_bytes_g, lat, (uint32_t)(n - n1st) * row_bytes_g, bar);
                    if (mirror) {
                        int gi = grow + RC - 3;
                        for (int q = 0; q < 3; ++q, ++gi) {  // row by row: the three rows may straddle the lattice end
                            if (!SLAB && gi >= (int)L) gi -= (int)L;
                            bulk_g2s(ring_s - (uint32_t)((3 - q) * pitch), lat + (ptrdiff_t)gi * (ptrdiff_t)row_bytes_g, row_bytes_g, bar);
                        }
                    }
                }
                __syncwarp();
                if (++slot == NR) { slot = 0; if (first_lap) first_lap = false; else par ^= 1u; }
                grow += RC;
                if (!SLAB && grow >= (int)L) grow -= (int)L;
            }
        }
    } else if (warp > kLeanConsumers) {
        // ---------------- packer warps (uint8 source): staging slots -> ring chunks ----------------
        // A pack iteration = 1024 staged bytes -> 128 ring bytes; slot rows are contiguous at pitch L
        // = (iterations per row) * 1024 and ring rows at pitch L/8, so both addresses are affine in it.
        if (SRC == kFmtU8) {
            const uint32_t pk = (uint32_t)(warp - kLeanConsumers - 1);
            const uint32_t lgIPR = g.lg2L - 10u;  // log2(1024-byte pack iterations per row)
            const uint32_t n_it = g.SR << lgIPR;
            uint32_t sslot = 0, spar = 0;         // staging slot to consume next, parity of its "full" barrier
            uint32_t rslot = 0, epar = 0;         // ring chunk to fill next, wait parity of its "empty" barrier
            bool first_lap = true;
            for (uint32_t c = 0; c < n_chunks; ++c) {
                if (!first_lap) mbar_wait_relaxed(bar_empty + 8u * rslot, epar);  // the workers are done with chunk c - NR
                const int dst_chunk = ring_off + (int)rslot * chunk_bytes + 2 * lane;
                const bool last_slot = rslot == NR - 1;  // its last three rows are mirrored in front of row 0
                for (uint32_t j = 0; j < g.SPC; ++j) {
                    const int r0 = (int)(j * g.SR);
                    if (c == 0 && r0 + (int)g.SR <= RC - 3) continue;  // never staged
                    mbar_wait_relaxed(bar_sfull + 8u * sslot, spar);
                    const uint8_t* src = smem_raw + (stage_off + (int)(sslot * g.slot_bytes) + 16 * lane) + (pk << 10);
                    uint8_t* dst = smem_raw + (dst_chunk + r0 * pitch) + (pk << 7);
                    // rows >= RC - 3 of a chunk start at iteration it_tail of their slot (chunk 0: only they are staged)
                    const int tail_rows = min((int)g.SR, max(0, r0 + (int)g.SR - (RC - 3)));
                    const uint32_t it_tail = (g.SR - (uint32_t)tail_rows) << lgIPR;
                    for (uint32_t it = pk; it < n_it; it += kLeanPackers, src += kLeanPackers * 1024, dst += kLeanPackers * 128) {
                        if (c == 0 && it < it_tail) continue;
                        const uint4 v0 = *reinterpret_cast<const uint4*>(src);
                        const uint4 v1 = *reinterpret_cast<const uint4*>(src + 512);
                        const uint16_t h0 = (uint16_t)lean_pack16(v0), h1 = (uint16_t)lean_pack16(v1);
                        *reinterpret_cast<uint16_t*>(dst) = h0;
                        *reinterpret_cast<uint16_t*>(dst + 64) = h1;
                        if (last_slot && it >= it_tail) {
                            *reinterpret_cast<uint16_t*>(dst - ring_bytes) = h0;
                            *reinterpret_cast<uint16_t*>(dst - ring_bytes + 64) = h1;
                        }
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive_cta(bar_sempty + 8u * sslot);  // my share of the slot is read
                    if (++sslot == g.NS) { sslot = 0; spar ^= 1u; }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive_cta(bar_full + 8u * rslot);  // my share of the chunk is in the ring
                if (++rslot == NR) { rslot = 0; if (first_lap) first_lap = false; else epar ^= 1u; }
            }
        }
    } else {
        // ---------------- worker warps ----------------
        const StepKey sk = make_step_key(a.seeds[b], a.t_begin + m, k, cls);
        uint2* q1 = reinterpret_cast<uint2*>(smem_raw + q_off + warp * kLeanWarpQBytes);
        uint4* q2 = reinterpret_cast<uint4*>(q1 + kLeanQ1Cap);
        const int colmask = (int)L - 1;
        const uint32_t cm = 0x11111111u << cj;  // the active sites of a 32-site word
        const uint32_t lt = (1u << lane) - 1u;
        uint32_t n1 = 0, n2 = 0, h2 = 0;
        int delta = 0;

        // ---- level 2 (a5-a7) on one Q2 entry (ring bit offset | dir << 30 | s_x << 29, site, u)
        auto level2 = [&](uint4 w) {
            const int soff = (int)(w.x & 0x1FFFFFFFu), sx = (int)((w.x >> 29) & 1u);
            const uint32_t dir = w.x >> 30;
            const int col = soff & colmask;
            int idx_t;
            if (GAME == kGamePD) {
                // n_x, n_y: the four neighbours of x and of y = x + e; columns wrap inside the row
                const int ps = colmask + 1, rowb = soff - col;
                auto N4 = [&](int rb, int c) {
                    return ring_get<kFmtBits>(ring0, rb - ps + c) + ring_get<kFmtBits>(ring0, rb + ps + c) +
                           ring_get<kFmtBits>(ring0, rb + ((c - 1) & colmask)) + ring_get<kFmtBits>(ring0, rb + ((c + 1) & colmask));
                };
                const int yr = rowb + (dir == 0u ? -ps : dir == 1u ? ps : 0);
                const int yc = (col + (dir == 2u ? -1 : dir == 3u ? 1 : 0)) & colmask;
                idx_t = sx * 25 + N4(rowb, col) * 5 + N4(yr, yc);
            } else {
                const int dA = (col < 3 || col > colmask - 3)
                                   ? ring_stencil_fr<kFmtBits>(soff, dir, sx, ring0, 0, colmask)
                                   : bits_stencil_lut(soff, dir, sx, reinterpret_cast<const uint32_t*>(ring0), pitch >> 2, lut);
                idx_t = sx * 102 + dA + 25;  // table_index(dA, ds) with ds = 2 s_x - 1
            }
            if (w.z < tbl[idx_t]) {
                if (SRC == kFmtU8)
                    lat[w.y] = (uint8_t)(1 - sx);
                else
                    atomicXor(reinterpret_cast<uint32_t*>(lat) + (w.y >> 5), 1u << (w.y & 31u));
                if (SLAB) {  // a boundary row of the slab is a halo row of a neighbour: push the new value
                    const int own = (int)(w.y >> g.lg2L) - (int)sl->row0, n_rows = (int)sl->n_rows, cx = (int)(w.y & (uint32_t)colmask);
                    if (own < 3) SlabLattice<SRC>::set(sl->up_halo, (int)L, own, cx, 1 - sx);
                    if (own >= n_rows - 3) SlabLattice<SRC>::set(sl->dn_halo, (int)L, own - (n_rows - 3), cx, 1 - sx);
                }
                delta += 1 - 2 * sx;
            }
        };
        auto run_level2 = [&](uint32_t cnt) {  // the first cnt (<= 32) entries of Q2
            if ((uint32_t)lane < cnt) level2(q2[(h2 + lane) & (kLeanQ2Cap - 1)]);
            __syncwarp();
            h2 += cnt;
            n2 -= cnt;
        };
        // ---- level 1 (a3, a4) on one Q1 entry; survivors are appended to Q2
        auto level1 = [&](uint2 e, uint4& w) -> bool {
            uint32_t x0, u;
            step_draw(sk, e.y, x0, u);
            const uint32_t dir = x0 >> 30;  // 0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1)
            const int soff = (int)e.x;
            const int sx = ring_get<kFmtBits>(ring0, soff);
            const int sy = ring_get<kFmtBits>(ring0, ring_nbr<true>(soff, dir, eoff[dir], colmask));
            w = make_uint4(e.x | (dir << 30) | ((uint32_t)sx << 29), e.y, u, 0u);
            return sx != sy;
        };
        auto push2 = [&](bool go, const uint4& w) {
            const uint32_t mk = __ballot_sync(0xFFFFFFFFu, go);
            if (go) q2[(h2 + n2 + __popc(mk & lt)) & (kLeanQ2Cap - 1)] = w;
            n2 += __popc(mk);
            __syncwarp();
            if (n2 >= 32u) run_level2(32u);
        };
        auto run_level1 = [&](uint32_t head, uint32_t cnt) {
            uint4 w;
            bool go = false;
            if ((uint32_t)lane < cnt) go = level1(q1[head + lane], w);
            push2(go, w);
        };
        // full batches from the front of Q1, two at a time while 64 wait (two independent Philox
        // chains); the leftover (< 32) moves to the front
        auto run_batches = [&]() {
            if (n1 < 64u) return;
            uint32_t head = 0;
            while (n1 - head >= 64u) {
                uint4 wa, wb;
                const bool ga = level1(q1[head + lane], wa);
                const bool gb = level1(q1[head + 32 + lane], wb);
                push2(ga, wa);
                push2(gb, wb);
                head += 64u;
            }
            const uint32_t left = n1 - head;  // < 64: waits for the next round, so that every batch runs in a pair
            uint2 e0 = make_uint2(0u, 0u), e1 = make_uint2(0u, 0u);
            if ((uint32_t)lane < left) e0 = q1[head + lane];
            if ((uint32_t)lane + 32u < left) e1 = q1[head + 32 + lane];
            __syncwarp();
            if ((uint32_t)lane < left) q1[lane] = e0;
            if ((uint32_t)lane + 32u < left) q1[32 + lane] = e1;
            __syncwarp();
            n1 = left;
        };
        // ---- survivors of one 32-site word per lane -> Q1, lane-serially after a warp prefix sum.
        // At most 128 new entries per round (Q1 holds 160): a crowded word goes in two halves.
        auto extract_round = [&](uint32_t z, uint32_t xb, uint32_t sb, bool may_split) {
            // prefix sum of the per-lane counts (0..8) from four ballots: the bits of the counts are summed
            // by population counts, all independent -- a shuffle scan is five dependent round trips
            const uint32_t cnt = __popc(z);
            const uint32_t b0 = ballot_bit<0>(cnt), b1 = ballot_bit<1>(cnt), b2 = ballot_bit<2>(cnt), b3 = ballot_bit<3>(cnt);
            const uint32_t tot = __reduce_add_sync(0xFFFFFFFFu, cnt);  // one REDUX instead of four POPC and three adds
            if (may_split && tot > 128u) return false;
            const uint32_t excl = __popc(b0 & lt) + 2u * __popc(b1 & lt) + 4u * __popc(b2 & lt) + 8u * __popc(b3 & lt);
            uint2* dst = q1 + n1 + excl;
            while (z) {  // two survivors per trip: the highest and the lowest set bit
                uint32_t hi;  // bfind = the position of the highest set bit (one FLO; 31 - __clz costs three)
                asm("bfind.u32 %0, %1;" : "=r"(hi) : "r"(z));
                const uint32_t lo = (uint32_t)__ffs((int)z) - 1u;
                dst[0] = make_uint2(xb + hi, sb + hi);
                if (hi != lo) dst[1] = make_uint2(xb + lo, sb + lo);
                dst += 2;  // (a lone last survivor leaves dst one too far: it is not used again)
                z = (z & (z - 1u)) & ~(1u << hi);  // drop the lowest and the highest set bit
            }
            __syncwarp();
            n1 += tot;
            run_batches();
            return true;
        };
        auto drain_all = [&]() {
            if (n1 > 32u) {  // < 64
                run_level1(0u, 32u);
                run_level1(32u, n1 - 32u);
                n1 = 0;
            } else if (n1) {
                run_level1(0u, n1);
                n1 = 0;
            }
            if (n2) run_level2(n2);  // < 32
        };

        if (n_steps) mbar_wait(bar_full, 0u);  // the tail of chunk 0
        const uint32_t lgWPR = g.lgWPR, wpr_mask = (1u << lgWPR) - 1u;
        const int wpitch = pitch >> 2;
        const uint32_t lag = g.lag, lag_mask = lag - 1u;
        uint32_t cslot = 1, fpar = 0;      // ring slot of chunk s + 1 and the parity of its "full" barrier
        int cur_off = chunk_bytes;         // = cslot * chunk_bytes
        uint32_t rel_slot = 0;             // ring slot of the next chunk to release
        uint32_t lat_row0 = 4u * (S0 * g.R) + (uint32_t)ci;  // lattice row of the step's first active row
        for (uint32_t s = 0; s < n_steps; ++s) {
            mbar_wait(bar_full + 8u * cslot, fpar);
            const uint32_t wrot = ((uint32_t)warp + s) & (kLeanConsumers - 1);  // column tasks rotate over the warps
            for (uint32_t seg = 0; seg < g.n_seg; ++seg) {
                const uint32_t W = seg * 512u + wrot * 32u + (uint32_t)lane;  // word of the step's R active rows
                const uint32_t rho = W >> lgWPR, kw = W & wpr_mask;
                const int rowb = cur_off + (int)rho * 4 * pitch;             // byte offset of the active row from ring0
                const uint32_t* rowp = reinterpret_cast<const uint32_t*>(ring0 + rowb);
                const uint32_t c = rowp[kw], u = rowp[(int)kw - wpitch], d = rowp[(int)kw + wpitch];
                const uint32_t pv = rowp[(kw - 1u) & wpr_mask], nx = rowp[(kw + 1u) & wpr_mask];
                const uint32_t lw = __funnelshift_l(pv, c, 1), rw = __funnelshift_r(c, nx, 1);
                const uint32_t nb = ((c ^ u) | (c ^ d) | (c ^ lw) | (c ^ rw)) & cm;  // S9
                if (__any_sync(0xFFFFFFFFu, nb != 0u)) {
                    const uint32_t xb = 8u * (uint32_t)rowb + 32u * kw;      // ring bit offset: ring rows are L bits
                    const uint32_t sb = ((lat_row0 + 4u * rho) << g.lg2L) + 32u * kw;
                    if (!extract_round(nb, xb, sb, true)) {
                        extract_round(nb & 0x0000FFFFu, xb, sb, false);
                        extract_round(nb & 0xFFFF0000u, xb, sb, false);
                    }
                }
            }
            // a queued site waits for at most `lag` steps: the ring keeps its rows that long
            if (((s + 1u) & lag_mask) == 0u) drain_all();
            if (s >= lag) {
                __syncwarp();
                if (lane == 0) mbar_arrive_cta(bar_empty + 8u * rel_slot);  // chunk s - lag is free
                if (++rel_slot == NR) rel_slot = 0;
            }
            lat_row0 += (uint32_t)RC;
            cur_off += chunk_bytes;
            if (++cslot == NR) { cslot = 0; fpar ^= 1u; cur_off = 0; }
        }
        drain_all();
        if (a.deltas != nullptr) {
            delta = __reduce_add_sync(0xFFFFFFFFu, delta);
            if (lane == 0 && delta != 0) atomicAdd(&delta_cta, delta);
        }
    }
    __syncthreads();
    if (a.deltas != nullptr && threadIdx.x == 0 && delta_cta != 0)
        atomicAdd(a.deltas + (size_t)b * a.n_mcs + m, (unsigned long long)(long long)delta_cta);
    // after the __syncthreads: every flip and push of this CTA is issued
    if (SLAB && threadIdx.x == 0) slab_post_edge(*sl, epoch, blockIdx.x == 0, blockIdx.x == gridDim.x - 1);
}

// One phase on a row slab (pgg_slab_sweep): LEAN's kernel on the slab's buffer, rows of layout SRC.
template <int SRC, int GAME = kGamePGG>
__global__ void __launch_bounds__(SRC == kFmtU8 ? kLeanThreadsU8 : kLeanThreads, 1)
phase_lean_slab_kernel(PhaseArgs a, uint32_t m, uint32_t k, LeanPlan g, SlabArgs sa, uint32_t epoch)
{
    lean_phase<SRC, GAME, false, true>(a, m, k, g, true, &sa, epoch);
}

template <int SRC, int GAME = kGamePGG>
__global__ void __launch_bounds__(SRC == kFmtU8 ? kLeanThreadsU8 : kLeanThreads, 1)
phase_lean_kernel(PhaseArgs a, uint32_t m, uint32_t k, LeanPlan g)
{
    lean_phase<SRC, GAME, false>(a, m, k, g);
}

// ---------------------------------------------------------------------------
// PERSIST: every phase of n_mcs MCS (16 n_mcs phases) in ONE cooperative launch, bit-packed source.
// ("minimizing the need to access global memory" -- and, on this machine, the launches.)
// The lattice stays where it is (L2-resident for the sizes this is used for).  A phase reads what the previous
// one wrote within radius 3 of every site, so a band (whole rows) waits, between two phases, for its TWO
// NEIGHBOUR bands only -- a flag per band in global memory, release / acquire at GPU scope; no grid-wide barrier,
// lattices of an ensemble never wait for each other.  What it saves is the launch, the drain of the grid and the
// refill of 148 empty pipelines behind a grid-wide dependency; what it costs is the flag round trip through L2
// and the set-up of a phase on the critical path (a dependent launch hides its set-up behind the previous
// phase's tail) -- measured slower than the launches (DESIGN.md appendix B): selectable, never AUTO.
// gbar[b * nb + band] = phases band `band` of lattice b has completed (zeroed by the host).
// ---------------------------------------------------------------------------
template <int GAME>
__global__ void __launch_bounds__(kLeanThreads, 1)
sweep_lean_kernel(PhaseArgs a, uint32_t m0, uint32_t n_mcs, LeanPlan g, unsigned int* __restrict__ gbar)
{
    const uint32_t n_phases = 16u * n_mcs;
    // done[band] = phases this band has completed.  A band reads its neighbours' three nearest rows and nothing
    // further, so phase p + 1 of band b needs phase p of bands b - 1, b, b + 1 only (both ways: they must also be
    // done READING b's rows of phase p before b changes them): neighbours are at most one phase apart, the rest
    // of the lattice may drift -- no grid-wide barrier, a slow band delays only its neighbourhood.
    unsigned int* done = gbar + (size_t)blockIdx.y * g.nb;
    const uint32_t band = blockIdx.x;
    const unsigned int* up = done + (band + g.nb - 1u) % g.nb;
    const unsigned int* dn = done + (band + 1u) % g.nb;
    for (uint32_t p = 0; p < n_phases; ++p) {
        lean_phase<kFmtBits, GAME, true>(a, m0 + (p >> 4), p & 15u, g, p == 0);  // ends with __syncthreads()
        if (p + 1 == n_phases) break;
        if (threadIdx.x == 0) {
            __threadfence();  // this CTA's flips (atomics) and counts before its flag
            const unsigned int target = p + 1u;
            asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(done + band), "r"(target) : "memory");
            unsigned int s0, s1, spins = 0;
            for (;;) {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(s0) : "l"(up) : "memory");
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(s1) : "l"(dn) : "memory");
                if (s0 >= target && s1 >= target) break;
                __nanosleep(20);
                if (++spins > (1u << 24)) __trap();  // ~1 s: a lost CTA must not hang the device
            }
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------
// PGG_VARIANT_PACKED: uint8 lattices <-> a bit-packed working copy (pure layout: bit j & 31 of word
// i (L/32) + (j >> 5) = byte (i, j), include/pgg.h).  One 32-site word per thread and trip: two 16-byte
// loads -> one 4-byte store, and back.  n_words = B L^2 / 32 over all lattices (they are contiguous in both).
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
pack_u8_kernel(const uint8_t* __restrict__ src, uint32_t* __restrict__ dst, unsigned long long n_words)
{
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long w = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; w < n_words; w += stride) {
        const uint4* p = reinterpret_cast<const uint4*>(src) + 2ull * w;
        const uint4 v0 = __ldcs(p), v1 = __ldcs(p + 1);  // read once: do not displace the working copy from L2
        dst[w] = (lean_pack16(v0) & 0xFFFFu) | (lean_pack16(v1) << 16);
    }
}

__global__ void __launch_bounds__(256)
unpack_u8_kernel(const uint32_t* __restrict__ src, uint8_t* __restrict__ dst, unsigned long long n_words)
{
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long w = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; w < n_words; w += stride) {
        const uint32_t v = src[w];
        uint32_t o[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {  // four sites per 32-bit word, one byte each
            const uint32_t nib = (v >> (4 * q)) & 0xFu;
            o[q] = (nib & 1u) | ((nib & 2u) << 7) | ((nib & 4u) << 14) | ((nib & 8u) << 21);
        }
        uint4* p = reinterpret_cast<uint4*>(dst) + 2ull * w;
        __stcs(p, make_uint4(o[0], o[1], o[2], o[3]));
        __stcs(p + 1, make_uint4(o[4], o[5], o[6], o[7]));
    }
}

inline void packed_launch(bool pack, uint8_t* d_u8, uint8_t* d_bits, unsigned long long n_words, cudaStream_t stream)
{
    const uint32_t grid = (uint32_t)std::min<unsigned long long>((n_words + 255ull) / 256ull, 148ull * 16ull);
    if (pack) pack_u8_kernel<<<grid, 256, 0, stream>>>(d_u8, reinterpret_cast<uint32_t*>(d_bits), n_words);
    else unpack_u8_kernel<<<grid, 256, 0, stream>>>(reinterpret_cast<const uint32_t*>(d_bits), d_u8, n_words);
}

// ---------------------------------------------------------------------------
// Host side
// ---------------------------------------------------------------------------
inline bool lean_supported(int /*fmt*/, uint32_t L)
{
    return L >= 1024 && L <= 32768 && (L & (L - 1)) == 0;  // whole 1024-byte pack units, power-of-two rows
}

inline int lean_plan(int fmt, uint32_t L, uint32_t B, LeanPlan* p)
{
    int dev = 0, sms = 0, smem_optin = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
    e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return (int)e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return (int)e;
    // per device and cheap next to the launches of a sweep: set on every plan
    e = cudaFuncSetAttribute((const void*)phase_lean_kernel<kFmtU8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 256);
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute((const void*)phase_lean_kernel<kFmtBits>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 256);
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute((const void*)phase_lean_kernel<kFmtU8, kGamePD>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 256);
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute((const void*)phase_lean_kernel<kFmtBits, kGamePD>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 256);
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute((const void*)sweep_lean_kernel<kGamePGG>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 256);
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute((const void*)sweep_lean_kernel<kGamePD>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 256);
    if (e != cudaSuccess) return (int)e;
    uint32_t lg = 0;
    while ((1u << lg) < L) ++lg;
    p->lg2L = lg;
    p->step0 = 0;
    p->pitch = L / 8;
    p->lgWPR = lg - 5;
    const uint32_t wpr = L / 32;
    p->R = wpr >= 512 ? 1u : 512u / wpr;
    p->n_seg = wpr > 512 ? wpr / 512 : 1u;
    uint32_t per_lat = (uint32_t)sms / B;
    if (per_lat < 1) per_lat = 1;
    // Two words per lane and step (R doubles) halve the per-step overhead: 46.5 against 50.4 us per phase on
    // bit-packed C5.  Only where a band keeps >= 8 steps (the ring fills once per band) and, for uint8, never:
    // there the doubled ring chunks squeeze the staging slots (77 against 64 us).
    uint32_t words = (fmt == kFmtBits && (L / 4) % (2 * p->R) == 0 && (L / 4) / (2 * p->R) >= 8 * per_lat) ? 2u : 1u;
    if (const char* s = getenv("PGG_LEAN_WORDS")) words = (atoi(s) == 2 && (L / 4) % (2 * p->R) == 0) ? 2u : 1u;
    if (words == 2) { p->R *= 2; p->n_seg *= 2; }
    p->RC = 4 * p->R;
    p->n_steps_total = (L / 4) / p->R;
    // (Two CTAs per SM fit the bit-packed ring, but need <= 60 registers per thread: the spills cost
    // more than the second CTA hides -- 46 against 40 us per phase, DESIGN.md appendix B.)
    p->nb = p->n_steps_total < per_lat ? p->n_steps_total : per_lat;
    const uint32_t avail = (uint32_t)smem_optin - 256 - kLeanFixedBytes;
    const uint32_t chunk_bits_bytes = p->RC * p->pitch;
    auto env_lag = [](uint32_t dflt) {
        if (const char* s = getenv("PGG_LEAN_LAG")) {
            const uint32_t v = (uint32_t)atoi(s);
            if (v >= 1 && v <= 16 && (v & (v - 1)) == 0) return v;
        }
        return dflt;
    };
    if (fmt == kFmtU8) {
        p->lag = env_lag(kLeanLagU8);
        uint32_t ahead = 2;  // ring chunks the packers may run ahead of the workers, beyond the lag + 3 the workers hold
        if (const char* s = getenv("PGG_LEAN_AHEAD")) ahead = (uint32_t)std::max(0, std::min(6, atoi(s)));
        while (p->lag > 1 && 3 * p->pitch + (p->lag + 3 + ahead) * chunk_bits_bytes + 2 * 32768u > avail) p->lag >>= 1;
        p->NR = std::min<uint32_t>(p->lag + 3 + ahead, kLeanMaxSlots);
        const uint32_t ring = 3 * p->pitch + p->NR * chunk_bits_bytes;
        uint32_t sr = 32768u / L;
        if (sr < 1) sr = 1;
        if (sr > p->RC) sr = p->RC;
        if (const char* s = getenv("PGG_LEAN_SLOT_ROWS")) {
            const uint32_t v = (uint32_t)atoi(s);
            if (v >= 1 && v <= p->RC && (p->RC % v) == 0 && v * L <= 65536u) sr = v;
        }
        p->SR = sr;
        p->SPC = p->RC / sr;
        p->slot_bytes = sr * L;
        if (ring + 2 * p->slot_bytes > avail) return (int)cudaErrorInvalidValue;
        uint32_t ns = (avail - ring) / p->slot_bytes;
        if (ns > (uint32_t)kLeanMaxSlots) ns = kLeanMaxSlots;
        if (const char* s = getenv("PGG_LEAN_SLOTS")) {
            const uint32_t v = (uint32_t)atoi(s);
            if (v >= 2 && v < ns) ns = v;
        }
        p->NS = ns;
        p->smem_bytes = ring + ns * p->slot_bytes + kLeanFixedBytes;
    } else {
        uint32_t nr = (avail - 3 * p->pitch) / chunk_bits_bytes;
        if (nr > (uint32_t)kLeanMaxSlots) nr = kLeanMaxSlots;
        p->lag = env_lag(kLeanLagBits);
        while (p->lag > 1 && p->lag + 3 > nr) p->lag >>= 1;
        if (nr < p->lag + 3) return (int)cudaErrorInvalidValue;
        p->NR = nr;
        p->SR = p->SPC = p->NS = p->slot_bytes = 0;
        p->smem_bytes = 3 * p->pitch + nr * chunk_bits_bytes + kLeanFixedBytes;
    }
    return 0;
}

inline void lean_launch(const LeanPlan& p, int fmt, const PhaseArgs& a, uint32_t m, uint32_t k, uint32_t B,
                        cudaStream_t stream, int game = kGamePGG)
{
    static const bool pdl = [] { const char* e = getenv("PGG_PDL"); return e == nullptr || atoi(e) != 0; }();
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(p.nb, B);
    cfg.blockDim = dim3(fmt == kFmtU8 ? kLeanThreadsU8 : kLeanThreads);
    cfg.dynamicSmemBytes = p.smem_bytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (game == kGamePD) {
        if (fmt == kFmtU8)
            cudaLaunchKernelEx(&cfg, phase_lean_kernel<kFmtU8, kGamePD>, a, m, k, p);
        else
            cudaLaunchKernelEx(&cfg, phase_lean_kernel<kFmtBits, kGamePD>, a, m, k, p);
    } else if (fmt == kFmtU8)
        cudaLaunchKernelEx(&cfg, phase_lean_kernel<kFmtU8>, a, m, k, p);
    else
        cudaLaunchKernelEx(&cfg, phase_lean_kernel<kFmtBits>, a, m, k, p);
}

// LEAN on a row slab: the geometry of the whole lattice (one bit-packed lattice of size L), the steps of the slab.
// Returns 0, or nonzero if the slab's rows are not whole steps (the caller takes the general slab kernel).
inline int lean_plan_slab(int fmt, uint32_t L, uint32_t row0, uint32_t n_rows, LeanPlan* p)
{
    if (!lean_supported(fmt, L)) return -1;
    int rc = lean_plan(fmt, L, 1, p);
    if (rc != 0) return rc;
    if ((n_rows / 4) % p->R != 0 || (row0 / 4) % p->R != 0) return -1;
    const void* fns[4] = {(const void*)phase_lean_slab_kernel<kFmtU8>, (const void*)phase_lean_slab_kernel<kFmtBits>,
                          (const void*)phase_lean_slab_kernel<kFmtU8, kGamePD>, (const void*)phase_lean_slab_kernel<kFmtBits, kGamePD>};
    cudaError_t e = cudaSuccess;
    for (const void* fn : fns)
        if ((e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->smem_bytes)) != cudaSuccess) return (int)e;
    int dev = 0, sms = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return (int)e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return (int)e;
    p->n_steps_total = (n_rows / 4) / p->R;
    p->step0 = (row0 / 4) / p->R;
    p->nb = p->n_steps_total < (uint32_t)sms ? p->n_steps_total : (uint32_t)sms;
    return 0;
}

inline void lean_slab_launch(const LeanPlan& p, int fmt, const PhaseArgs& a, uint32_t m, uint32_t k, const SlabArgs& sa,
                             uint32_t epoch, cudaStream_t stream, int game = kGamePGG)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(p.nb, 1);
    cfg.blockDim = dim3(fmt == kFmtU8 ? kLeanThreadsU8 : kLeanThreads);
    cfg.dynamicSmemBytes = p.smem_bytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (game == kGamePD) {
        if (fmt == kFmtU8)
            cudaLaunchKernelEx(&cfg, phase_lean_slab_kernel<kFmtU8, kGamePD>, a, m, k, p, sa, epoch);
        else
            cudaLaunchKernelEx(&cfg, phase_lean_slab_kernel<kFmtBits, kGamePD>, a, m, k, p, sa, epoch);
    } else if (fmt == kFmtU8)
        cudaLaunchKernelEx(&cfg, phase_lean_slab_kernel<kFmtU8>, a, m, k, p, sa, epoch);
    else
        cudaLaunchKernelEx(&cfg, phase_lean_slab_kernel<kFmtBits>, a, m, k, p, sa, epoch);
}

// One cooperative launch for MCS [m0, m0 + n_mcs) of B lattices; d_gbar: B zeroed counters.
inline cudaError_t lean_persist_launch(const LeanPlan& p, const PhaseArgs& a, uint32_t m0, uint32_t n_mcs, uint32_t B,
                                       unsigned int* d_gbar, cudaStream_t stream, int game = kGamePGG)
{
    PhaseArgs a_ = a;
    LeanPlan p_ = p;
    void* args[] = {&a_, &m0, &n_mcs, &p_, &d_gbar};
    const void* fn = game == kGamePD ? (const void*)sweep_lean_kernel<kGamePD> : (const void*)sweep_lean_kernel<kGamePGG>;
    return cudaLaunchCooperativeKernel(fn, dim3(p.nb, B), dim3(kLeanThreads), args, p.smem_bytes, stream);
}

// Can the persistent kernel run this workload?  Bit-packed, and every CTA resident at once.
inline bool lean_persist_supported(int fmt, uint32_t L, uint32_t B)
{
    return fmt == kFmtBits && lean_supported(fmt, L) && B <= 148;
}

}  // namespace pgg
