// pgg_kernels_cluster.cuh -- the CLUSTER kernel: one lattice of L = 128 .. 4096 (a power of two) stays BIT-PACKED in
// the shared memory of a thread-block cluster for a whole call ("minimizing
// the need to access global memory, and to make full use of the registers and the shared memory").
//
// Round-2 measurements (appendix B): a phase of an L2-resident lattice costs 4-5 us
// whatever it contains -- the latency of class lookup -> bulk copy -> L2 round trip -> one step -> drain
// -- and neither fewer bytes (LEAN) nor fewer launches (PERSIST) shorten that chain.  Keeping the rows
// on chip does: nothing is staged, nothing waits for a copy, and the queues are drained once per phase.
//
//   cluster  = CS CTAs (1 .. 16, from L and the number of lattices; 16 is a non-portable size) = one lattice; grid = (CS, B)
//   band     = the L/CS consecutive rows CTA `rank` owns, plus three halo rows above and below, all in
//              its shared memory as bits (uint8 lattices are packed on load and unpacked on store:
//              the layout in HBM is the caller's, the layout on chip is ours)
//   phase    = every worker lane scans one 32-site word of an active row per round (512 words per
//              round and CTA), survivors -> Q1 -> Philox on dense batches -> Q2 -> stencil on dense
//              batches, as LEAN's workers; flips are atomicXor on the CTA's own shared memory; the
//              queues are drained at the END of the phase (the rows never leave)
//   exchange = neighbours only, no cluster-wide barrier and no fence.  A phase of class row ci changes, of the rows a
//              neighbour mirrors, one row at most per side: row ci of the first three (ci <= 2) and row rows-4+ci of
//              the last three (ci >= 1).  After the CTA's own __syncthreads the owners of those words send them into
//              the neighbour's halo with st.async (SASS STAS), whose bytes count on the NEIGHBOUR's mbarrier; thread 0
//              adds a relaxed remote arrival "done with phase p".  Every thread then waits on its two halo barriers
//              (from above / from below; two per side, alternating with the phase, armed two phases ahead with the
//              bytes to expect).  Neighbours are at most one phase apart.  A row that arrives one phase early differs
//              from what was there only in sites of that phase's class, which no site reads during it (same-class
//              sites are >= 4 apart, reads reach 3: S1) -- the argument that makes the in-place update legal in the
//              first place.  Round-2 measurement: cluster.sync() compiled to MEMBAR.ALL.GPU + cluster barrier +
//              CCTL.IVALL in every thread and was the top stall (profiles/r2_ncu_full.md); without it a phase of one
//              1024^2 lattice takes 2.31 us instead of 2.72.
//   trace    = signed flip counts per CTA and MCS, one 64-bit atomic per CTA and MCS (a8)
// Clusters are independent: an ensemble larger than the GPU holds at once simply runs in waves.
#pragma once
#include <cooperative_groups.h>

#include "pgg_kernels_lean.cuh"

namespace pgg {

namespace cg = cooperative_groups;

constexpr int kClusterWarps = 16;
constexpr int kClusterThreads = kClusterWarps * 32;
constexpr int kClusterFixedBytes = kClusterWarps * kLeanWarpQBytes + 160 * 4 + 8 * 4 + kStencilLutBytes + 128;

struct ClusterPlan {
    uint32_t lg2L;
    uint32_t pitch;    // bytes per row = L / 8
    uint32_t lgWPR;    // log2(words per row)
    uint32_t CS;       // CTAs per cluster = bands per lattice
    uint32_t rows;     // rows per band = L / CS (a multiple of 4)
    uint32_t words_per_phase;  // (rows / 4) * (L / 32): a multiple of 32 (whole warps)
    uint32_t smem_bytes;
};

// ---- distributed shared memory: addresses of a neighbour CTA, asynchronous stores, remote barrier arrivals
__device__ __forceinline__ uint32_t cluster_map(uint32_t saddr, uint32_t cta_rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(cta_rank));
    return r;
}
// one 32-bit word into a neighbour's shared memory; its 4 bytes are counted on the neighbour's mbarrier (no fence needed)
__device__ __forceinline__ void st_async_b32(uint32_t raddr, uint32_t val, uint32_t rbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];" ::"r"(raddr), "r"(val), "r"(rbar) : "memory");
}
// "This CTA is done with the phase" on a neighbour's barrier.  Relaxed on purpose: the arrival orders nothing that is
// still in flight -- it tells the neighbour that this CTA's READS of its halo rows are over, and they are: every warp
// has used the values it read and passed __syncthreads before thread 0 gets here.  (A release at cluster scope costs
// MEMBAR.ALL.GPU on the critical path of every phase; the rows themselves travel by st.async, which needs no fence.)
__device__ __forceinline__ void mbar_arrive_remote(uint32_t rbar)
{
    asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(rbar) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!done);
}

template <int SRC, int GAME>
__global__ void __launch_bounds__(kClusterThreads, 1)
sweep_cluster_kernel(PhaseArgs a, uint32_t m0, uint32_t n_mcs, ClusterPlan g)
{
    extern __shared__ __align__(128) uint8_t smem_raw[];
    cg::cluster_group cluster = cg::this_cluster();
    const uint32_t rank = cluster.block_rank(), CS = g.CS;
    const uint32_t b = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t L = a.L, rows = g.rows;
    const int pitch = (int)g.pitch, wpr = pitch >> 2;
    uint8_t* ring0 = smem_raw + 3 * pitch;                       // own row 0; rows -3..-1 and rows..rows+2 are halos
    uint32_t* words = reinterpret_cast<uint32_t*>(smem_raw);      // word 0 = halo row -3
    const int q_off = (int)(rows + 6) * pitch;
    uint32_t* tbl = reinterpret_cast<uint32_t*>(smem_raw + q_off + kClusterWarps * kLeanWarpQBytes);
    int* eoff = reinterpret_cast<int*>(tbl + 160);
    int8_t* lut = reinterpret_cast<int8_t*>(eoff + 8);  // StencilLut (pgg_kernels_lean.cuh)
    __shared__ int delta_cta;
    // halo barriers [from above | from below][phase parity]: one phase of one of them = my own arming arrival (with the
    // bytes to expect) + the neighbour's "done" arrival + the bytes of the neighbour's changed row
    __shared__ __align__(8) unsigned long long xbar[4];
    uint8_t* lat = a.lats + (size_t)b * a.lat_bytes;
    const uint32_t n_phases = 16u * n_mcs;
    const uint32_t xbar_s = smem_u32(xbar);
    auto class_row = [&](uint32_t q) -> uint32_t {  // i mod 4 of the class of phase q of this call
        const uint32_t mq = m0 + (q >> 4);
        return (uint32_t)a.order[((size_t)b * a.order_stride + (mq % a.order_stride)) * 16 + (q & 15u)] >> 2;
    };
    // A phase of class row ci changes, of the rows a neighbour mirrors, only row ci of my first three (ci <= 2: the lower
    // halo of the band above) and row rows-4+ci of my last three (ci >= 1: the upper halo of the band below)
    auto arm = [&](uint32_t q) {
        const uint32_t ciq = class_row(q), par = q & 1u, row_bytes = 4u * (uint32_t)wpr;
        if (ciq >= 1u) mbar_expect_tx(xbar_s + 8u * par, row_bytes); else mbar_arrive_cta(xbar_s + 8u * par);
        if (ciq <= 2u) mbar_expect_tx(xbar_s + 8u * (2u + par), row_bytes); else mbar_arrive_cta(xbar_s + 8u * (2u + par));
    };
    if (threadIdx.x == 0) {
        for (int q = 0; q < 4; ++q) mbar_init(xbar_s + 8u * q, 2);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        arm(0u);
        arm(1u);  // n_phases >= 16
    }

    // ---- load the band and its halos (periodic rows), packing uint8 to bits
    const uint32_t n_words = (rows + 6u) * (uint32_t)wpr;
    const uint32_t row_first = rank * rows + L - 3u;             // lattice row of halo row -3 (mod L)
    for (uint32_t idx = threadIdx.x; idx < n_words; idx += kClusterThreads) {
        const uint32_t r = idx >> g.lgWPR, kw = idx & ((1u << g.lgWPR) - 1u);
        const uint32_t gi = (row_first + r) & (L - 1u);
        uint32_t w;
        if (SRC == kFmtU8) {
            const uint4* src = reinterpret_cast<const uint4*>(lat + (size_t)gi * L + 32u * kw);
            w = (lean_pack16(src[0]) & 0xFFFFu) | (lean_pack16(src[1]) << 16);
        } else {
            w = reinterpret_cast<const uint32_t*>(lat)[(size_t)gi * (uint32_t)wpr + kw];
        }
        words[idx] = w;
    }
    for (int q = threadIdx.x; q < kTableSize; q += kClusterThreads) tbl[q] = a.tables[(size_t)b * kTableSize + q];
    if (GAME == kGamePGG)
        for (int q = threadIdx.x; q < kStencilLutBytes / 4; q += kClusterThreads)
            reinterpret_cast<uint32_t*>(lut)[q] = reinterpret_cast<const uint32_t*>(g_stencil_lut.v)[q];
    if (threadIdx.x == 0) {
        delta_cta = 0;
        const int ps = (int)L;  // one row down, in bits
        eoff[0] = -ps; eoff[1] = ps; eoff[2] = -1; eoff[3] = 1;
        eoff[4] = 1;   eoff[5] = 1;  eoff[6] = ps; eoff[7] = ps;
    }
    __syncthreads();
    cluster.sync();  // every CTA of the cluster runs and has its rows before anyone stores into a neighbour

    // the neighbours' halo rows and halo barriers, as distributed-shared-memory addresses
    const uint32_t up = (rank + CS - 1u) % CS, dn = (rank + 1u) % CS, words_s = smem_u32(words);
    const uint32_t up_halo_bot = cluster_map(words_s + 4u * (rows + 3u) * (uint32_t)wpr, up);  // rows..rows+2 of the band above
    const uint32_t dn_halo_top = cluster_map(words_s, dn);                                     // rows -3..-1 of the band below
    const uint32_t up_bar = cluster_map(xbar_s + 16u, up), dn_bar = cluster_map(xbar_s, dn);   // its "from below" / "from above" pair

    uint2* q1 = reinterpret_cast<uint2*>(smem_raw + q_off + warp * kLeanWarpQBytes);
    uint4* q2 = reinterpret_cast<uint4*>(q1 + kLeanQ1Cap);
    const int colmask = (int)L - 1;
    const uint32_t lt = (1u << lane) - 1u;
    const uint32_t lgWPR = g.lgWPR, wpr_mask = (1u << lgWPR) - 1u;
    const uint64_t seed = a.seeds[b];
    uint32_t n1 = 0, n2 = 0, h2 = 0;
    int delta = 0;  // this lane's flips in the current MCS

    for (uint32_t p = 0; p < n_phases; ++p) {
        const uint32_t m = m0 + (p >> 4), k = p & 15u;
        const uint32_t cls = a.order[((size_t)b * a.order_stride + (m % a.order_stride)) * 16 + k];
        const int ci = (int)(cls >> 2), cj = (int)(cls & 3u);
        const StepKey sk = make_step_key(seed, a.t_begin + m, k, cls);
        const uint32_t cm = 0x11111111u << cj;  // the active sites of a 32-site word

        // ---- level 2 (a5-a7) on one Q2 entry (bit offset from own row 0 | dir << 30 | s_x << 29, site, u)
        auto level2 = [&](uint4 w) {
            const int soff = (int)(w.x & 0x1FFFFFFFu), sx = (int)((w.x >> 29) & 1u);
            const uint32_t dir = w.x >> 30;
            const int col = soff & colmask;
            int idx_t;
            if (GAME == kGamePD) {
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
                                   : bits_stencil_lut(soff, dir, sx, reinterpret_cast<const uint32_t*>(ring0), wpr, lut);
                idx_t = sx * 102 + dA + 25;
            }
            if (w.z < tbl[idx_t]) {
                atomicXor(reinterpret_cast<uint32_t*>(ring0) + (soff >> 5), 1u << (soff & 31));  // the CTA's own rows
                delta += 1 - 2 * sx;
            }
        };
        auto run_level2 = [&](uint32_t cnt) {
            if ((uint32_t)lane < cnt) level2(q2[(h2 + lane) & (kLeanQ2Cap - 1)]);
            __syncwarp();
            h2 += cnt;
            n2 -= cnt;
        };
        auto level1 = [&](uint2 e, uint4& w) -> bool {
            uint32_t x0, u;
            step_draw(sk, e.y, x0, u);
            const uint32_t dir = x0 >> 30;
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
        auto run_batches = [&]() {  // every batch in an interleaved pair; up to 63 entries wait (as in LEAN)
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
            const uint32_t left = n1 - head;
            uint2 e0 = make_uint2(0u, 0u), e1 = make_uint2(0u, 0u);
            if ((uint32_t)lane < left) e0 = q1[head + lane];
            if ((uint32_t)lane + 32u < left) e1 = q1[head + 32 + lane];
            __syncwarp();
            if ((uint32_t)lane < left) q1[lane] = e0;
            if ((uint32_t)lane + 32u < left) q1[32 + lane] = e1;
            __syncwarp();
            n1 = left;
        };
        auto extract_round = [&](uint32_t z, uint32_t xb, uint32_t sb, bool may_split) {
            const uint32_t cnt = __popc(z);
            const uint32_t b0 = ballot_bit<0>(cnt), b1 = ballot_bit<1>(cnt), b2 = ballot_bit<2>(cnt), b3 = ballot_bit<3>(cnt);
            const uint32_t tot = __reduce_add_sync(0xFFFFFFFFu, cnt);  // one REDUX instead of four POPC and three adds
            if (may_split && tot > 128u) return false;
            const uint32_t excl = __popc(b0 & lt) + 2u * __popc(b1 & lt) + 4u * __popc(b2 & lt) + 8u * __popc(b3 & lt);
            uint2* dst = q1 + n1 + excl;
            while (z) {
                uint32_t hi;  // bfind = the position of the highest set bit (one FLO; 31 - __clz costs three)
                asm("bfind.u32 %0, %1;" : "=r"(hi) : "r"(z));
                const uint32_t lo = (uint32_t)__ffs((int)z) - 1u;
                dst[0] = make_uint2(xb + hi, sb + hi);
                if (hi != lo) dst[1] = make_uint2(xb + lo, sb + lo);
                dst += 2;
                z = (z & (z - 1u)) & ~(1u << hi);  // drop the lowest and the highest set bit
            }
            __syncwarp();
            n1 += tot;
            run_batches();
            return true;
        };

        // ---- the phase: rounds of 512 words over the band's active rows
        for (uint32_t w0 = (uint32_t)warp * 32u + (uint32_t)lane; w0 < g.words_per_phase; w0 += kClusterThreads) {
            const uint32_t rho = w0 >> lgWPR, kw = w0 & wpr_mask;
            const int lrow = 4 * (int)rho + ci;                                    // row of the band
            const uint32_t* rowp = reinterpret_cast<const uint32_t*>(ring0 + lrow * pitch);
            const uint32_t c = rowp[kw], u = rowp[(int)kw - wpr], d = rowp[(int)kw + wpr];
            const uint32_t pv = rowp[(kw - 1u) & wpr_mask], nx = rowp[(kw + 1u) & wpr_mask];
            const uint32_t lw = __funnelshift_l(pv, c, 1), rw = __funnelshift_r(c, nx, 1);
            const uint32_t nb = ((c ^ u) | (c ^ d) | (c ^ lw) | (c ^ rw)) & cm;  // S9
            if (__any_sync(0xFFFFFFFFu, nb != 0u)) {
                const uint32_t xb = ((uint32_t)lrow << g.lg2L) + 32u * kw;
                const uint32_t sb = ((rank * rows + (uint32_t)lrow) << g.lg2L) + 32u * kw;
                if (!extract_round(nb, xb, sb, true)) {
                    extract_round(nb & 0x0000FFFFu, xb, sb, false);
                    extract_round(nb & 0xFFFF0000u, xb, sb, false);
                }
            }
        }
        if (n1 > 32u) {  // < 64
            run_level1(0u, 32u);
            run_level1(32u, n1 - 32u);
            n1 = 0;
        } else if (n1) {
            run_level1(0u, n1);
            n1 = 0;
        }
        if (n2) run_level2(n2);  // < 32
        if (k == 15u && a.deltas != nullptr) {  // a8: this MCS's flips of the whole CTA
            const int dw = __reduce_add_sync(0xFFFFFFFFu, delta);
            if (lane == 0 && dw != 0) atomicAdd(&delta_cta, dw);
            delta = 0;
        }
        __syncthreads();  // the CTA's flips of this phase are in its rows
        if (k == 15u && a.deltas != nullptr && threadIdx.x == 0 && delta_cta != 0) {
            atomicAdd(a.deltas + (size_t)b * a.n_mcs + m, (unsigned long long)(long long)delta_cta);
            delta_cta = 0;
        }
        // ---- exchange with the two neighbours only (no cluster-wide barrier, no fence): the one row of my first / last
        // three that this phase changed goes into their halo by asynchronous stores that count on THEIR barrier; thread 0
        // adds "this CTA is done with phase p" (every warp has passed the barrier above, so nobody here still reads the
        // halos of phase p: the neighbour may overwrite them with phase p+1).  Then everybody waits for the neighbours'
        // rows and "done".  Skew between neighbours is at most one phase, and a row that arrives one phase early differs
        // only in sites of that phase's class, which nobody reads during it (as for the in-place update itself).
        const uint32_t par = p & 1u;
        if (ci <= 2 && threadIdx.x < (uint32_t)wpr)
            st_async_b32(up_halo_bot + 4u * ((uint32_t)(ci * wpr) + threadIdx.x), words[(3 + ci) * wpr + (int)threadIdx.x], up_bar + 8u * par);
        if (ci >= 1 && threadIdx.x >= 256u && threadIdx.x < 256u + (uint32_t)wpr) {
            const uint32_t t = threadIdx.x - 256u;
            st_async_b32(dn_halo_top + 4u * ((uint32_t)((ci - 1) * wpr) + t), words[((int)rows + ci - 1) * wpr + (int)t], dn_bar + 8u * par);
        }
        if (threadIdx.x == 0) {
            mbar_arrive_remote(up_bar + 8u * par);
            mbar_arrive_remote(dn_bar + 8u * par);
        }
        const uint32_t use_par = (p >> 1) & 1u;
        mbar_wait_cluster(xbar_s + 8u * par, use_par);
        mbar_wait_cluster(xbar_s + 8u * (2u + par), use_par);
        if (threadIdx.x == 0 && p + 2u < n_phases) arm(p + 2u);
    }

    // ---- store the band back in the caller's layout
    const uint32_t own_words = rows * (uint32_t)wpr;
    for (uint32_t idx = threadIdx.x; idx < own_words; idx += kClusterThreads) {
        const uint32_t r = idx >> g.lgWPR, kw = idx & wpr_mask;
        const uint32_t gi = rank * rows + r;
        const uint32_t w = words[3 * wpr + idx];
        if (SRC == kFmtU8) {
            uint4* dst = reinterpret_cast<uint4*>(lat + (size_t)gi * L + 32u * kw);
            uint32_t o[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) {  // four sites per 32-bit word, one byte each
                const uint32_t nib = (w >> (4 * q)) & 0xFu;
                o[q] = (nib & 1u) | ((nib & 2u) << 7) | ((nib & 4u) << 14) | ((nib & 8u) << 21);
            }
            dst[0] = make_uint4(o[0], o[1], o[2], o[3]);
            dst[1] = make_uint4(o[4], o[5], o[6], o[7]);
        } else {
            reinterpret_cast<uint32_t*>(lat)[(size_t)gi * (uint32_t)wpr + kw] = w;
        }
    }
}

// ---------------------------------------------------------------------------
// Host side
// ---------------------------------------------------------------------------
inline bool cluster_supported(int /*fmt*/, uint32_t L)
{
    return L >= 128 && L <= 4096 && (L & (L - 1)) == 0;  // whole 32-site words, power-of-two rows, fits 16 CTAs
}

inline int cluster_plan(int fmt, uint32_t L, uint32_t B, ClusterPlan* p)
{
    uint32_t lg = 0;
    while ((1u << lg) < L) ++lg;
    p->lg2L = lg;
    p->pitch = L / 8;
    p->lgWPR = lg - 5;
    int dev = 0, smem_optin = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
    e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return (int)e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return (int)e;
    // CTAs per lattice.  Measured (DESIGN.md appendix B): a phase costs ~1.7 us + ~1.1 us per round of 512
    // words, so a lattice wants as many CTAs as give it half a round each -- as long as every lattice's
    // cluster is resident at once (the occupancy query knows how many clusters of a size the GPCs hold);
    // a larger ensemble takes the smallest cluster that fits shared memory and runs in waves.
    auto fits = [&](uint32_t cs) { return (L / cs) % 4 == 0 && (L / cs + 6) * p->pitch + (uint32_t)kClusterFixedBytes <= (uint32_t)smem_optin; };
    const void* k0 = fmt == kFmtU8 ? (const void*)sweep_cluster_kernel<kFmtU8, kGamePGG> : (const void*)sweep_cluster_kernel<kFmtBits, kGamePGG>;
    cudaFuncSetAttribute(k0, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    auto resident = [&](uint32_t cs) -> uint32_t {   // clusters of size cs the device holds at once
        const uint32_t smem = (L / cs + 6) * p->pitch + (uint32_t)kClusterFixedBytes;
        if (cudaFuncSetAttribute(k0, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return 0;
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(cs, B);
        cfg.blockDim = dim3(kClusterThreads);
        cfg.dynamicSmemBytes = smem;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = cs;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        int n = 0;
        if (cudaOccupancyMaxActiveClusters(&n, k0, &cfg) != cudaSuccess) { cudaGetLastError(); return 0; }
        return (uint32_t)n;
    };
    uint32_t cs_max = 2 * (L / 128) * (L / 512);   // half a round per CTA: 2 L^2 / 65536
    if (cs_max < 1) cs_max = 1;
    if (cs_max > 16) cs_max = 16;
    // cost model: waves x (1.7 us + 1.1 us per round); ties go to the smaller cluster
    uint32_t cs = 0;
    double best = 0.0;
    for (uint32_t c = 1; c <= cs_max; c <<= 1) {
        if (!fits(c)) continue;
        const uint32_t res = resident(c);
        if (res == 0) continue;
        const double rounds = (double)L * L / (65536.0 * c);
        const double cost = (double)((B + res - 1) / res) * (1.7 + 1.1 * (rounds < 0.5 ? 0.5 : rounds));
        if (cs == 0 || cost < 0.97 * best) { cs = c; best = cost; }
    }
    if (const char* s = getenv("PGG_CLUSTER_SIZE")) {
        const uint32_t v = (uint32_t)atoi(s);
        if ((v == 1 || v == 2 || v == 4 || v == 8 || v == 16) && fits(v)) cs = v;
    }
    if (cs == 0) return (int)cudaErrorInvalidValue;
    p->CS = cs;
    p->rows = L / p->CS;
    p->words_per_phase = (p->rows / 4) * (L / 32);   // a multiple of 32: whole warps
    p->smem_bytes = (p->rows + 6) * p->pitch + kClusterFixedBytes;
    const void* kernels[4] = {(const void*)sweep_cluster_kernel<kFmtU8, kGamePGG>, (const void*)sweep_cluster_kernel<kFmtBits, kGamePGG>,
                              (const void*)sweep_cluster_kernel<kFmtU8, kGamePD>, (const void*)sweep_cluster_kernel<kFmtBits, kGamePD>};
    for (const void* kern : kernels) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->smem_bytes);
        if (e != cudaSuccess) return (int)e;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return (int)e;
    }
    (void)fmt;
    return 0;
}

inline cudaError_t cluster_launch(const ClusterPlan& p, int fmt, const PhaseArgs& a, uint32_t m0, uint32_t n_mcs, uint32_t B,
                                  cudaStream_t stream, int game = kGamePGG)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(p.CS, B);
    cfg.blockDim = dim3(kClusterThreads);
    cfg.dynamicSmemBytes = p.smem_bytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = p.CS;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (game == kGamePD)
        return fmt == kFmtU8 ? cudaLaunchKernelEx(&cfg, sweep_cluster_kernel<kFmtU8, kGamePD>, a, m0, n_mcs, p)
                             : cudaLaunchKernelEx(&cfg, sweep_cluster_kernel<kFmtBits, kGamePD>, a, m0, n_mcs, p);
    return fmt == kFmtU8 ? cudaLaunchKernelEx(&cfg, sweep_cluster_kernel<kFmtU8, kGamePGG>, a, m0, n_mcs, p)
                         : cudaLaunchKernelEx(&cfg, sweep_cluster_kernel<kFmtBits, kGamePGG>, a, m0, n_mcs, p);
}

}  // namespace pgg
