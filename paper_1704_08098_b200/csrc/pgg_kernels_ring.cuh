// pgg_kernels_ring.cuh -- the RING phase kernel (K1 uint8, K2 bit-packed): the
// BAND kernel's data movement with a consumer path cut down to the fewest
// instructions.
//
// ncu on BAND at L = 16384 (profiles/r1_band_u8_late.md): the kernel is bound by
// instruction issue, not by HBM -- 56 M warp instructions per phase, 65 % issue
// utilisation, 83 us against the 44 us an HBM-bound pass would take; Philox is
// under 10 % of them, the rest is queue bookkeeping, address arithmetic of the
// generic (parity, ring row, column) queue entries, and the ring-wrap fix-up of
// every stencil access.  RING removes that work:
//
//   * a stencil access is ring0[soff + constant]; only sites in ring row 0 (one
//     step in NS) can reach above the ring, and only they take a second copy of
//     the stencil code whose negative offsets get the ring size added.  (The
//     alternative, PGG_RING_MIRROR=1, stages the three rows above slot 0 a second
//     time in front of it -- no wrap at all, but 24 KB that a sixth ring slot
//     uses better: 65.0 -> 63.5 us per launch, DESIGN.md appendix A);
//   * queue entries are self-contained: Q1 = (soff, site), Q2 = (soff|dir|s_x,
//     site, u); soff = offset of x from ring0 in site units (bytes for uint8,
//     bits for bit-packed), site = lattice site index (the Philox counter and
//     the address of the in-place write).  No parity / row decoding;
//   * the direction-dependent stencil offsets come from two 4-entry tables in
//     shared memory: e = step towards y, f = perpendicular step; the 14 reads of
//     A_x - A_y are ring0[soff + a e + b f] with six row bases shared between
//     them;
//   * level 1 runs two batches of 32 queued sites at once when 64 are waiting,
//     so two independent Philox chains hide each other's multiply latency;
//   * uint8 runs the stencil inline on the lanes whose drawn neighbour differs
//     (a second queue fills its batches only half: a site may wait one step
//     only); the bit-packed instantiation keeps Q2;
//   * launches carry the programmatic-dependent-launch attribute: a CTA sets up
//     while the previous phase drains and executes griddepcontrol.wait before it
//     touches the lattice;
//   * the 16 column tasks of a step rotate over the warps, so that no warp is
//     tied to the busiest columns of the band;
//   * full-row mode (FR): when the strip is the whole lattice row the halo
//     columns are dropped and a chunk arrives as ONE bulk copy;
//   * while it waits for the previous phase to drain (before griddepcontrol.wait)
//     the producer warp prefetches the band's first rows into L2.
//
// Geometry, producer, barriers and the compaction (scan -> Q1 -> Philox
// [-> Q2] -> stencil) are those of pgg_kernels_band.cuh:
//
//   strip  = W = tpr * 512 bytes of every lattice row (+ 16-byte halo each side)
//   band   = the consecutive lattice rows of a strip one persistent CTA streams
//   chunk  = RC = 4 R consecutive rows (R = 16 / tpr active rows), one ring slot
//   step s = the R active rows of chunk s + 1; reads reach the tail of chunk s
//   16 consumer warps (warp w: active row w / tpr, column task w % tpr) + 1
//   producer warp; chunk s - 1 is released at the end of step s, after every
//   site queued in step s - 1 has been finished.
#pragma once
#include "pgg_kernels_band.cuh"

namespace pgg {

constexpr int kRingConsumers = 16;
constexpr int kRingThreads = (kRingConsumers + 1) * 32;
constexpr int kRingTaskB = 512;   // bytes of one lattice row that one warp scans per step
constexpr int kRingHaloB = 16;
constexpr int kRingQ1Cap = 160;   // 8-byte entries per warp: leftover (< 32) + 128 new
constexpr int kRingQ2Cap = 64;    // 16-byte entries per warp (a ring: power of two)
constexpr int kRingMaxSlots = 6;
// Q2 (a second compaction between the Philox draw and the stencil) fills its batches of 32
// only half on average -- a site may wait for one step only -- and its 16 KB are worth more
// as ring slots (DESIGN.md appendix A), so level 2 runs inline under divergence.
// The bit-packed stencil (a shift and a mask per read) is dearer, there Q2 still pays.
template <int FMT> struct RingCfg {
    static constexpr bool q2 = FMT == kFmtBits;
    static constexpr int warp_q_bytes = kRingQ1Cap * 8 + (q2 ? kRingQ2Cap * 16 : 0);
    static constexpr int fixed_bytes = kRingConsumers * warp_q_bytes + 160 * 4 + 2 * kRingMaxSlots * 8 + 8 * 4 + 128;
};

struct RingPlan {
    uint32_t row_bytes;  // bytes per lattice row
    uint32_t W;          // strip width in bytes = tpr * 512
    uint32_t n_strips;
    uint32_t tpr_log2;   // log2(column tasks per row of a strip)
    uint32_t R;          // active rows per step = 16 / tpr
    uint32_t RC;         // lattice rows per chunk = 4 R
    uint32_t pitch;      // bytes per staged row = W + 32
    uint32_t slot_bytes; // RC * pitch
    uint32_t NS;         // ring slots
    uint32_t nb;         // bands (CTAs) per strip
    uint32_t n_groups;   // L / 4 active rows per class
    uint32_t n_super;    // steps per strip = ceil(n_groups / R)
    uint32_t smem_bytes;
    uint32_t mirror;     // 1: three mirror rows in front of slot 0; 0: wrapping stencil reads
    uint32_t rotate;     // 1: column tasks rotate over the warps from step to step
    uint32_t fullrow;    // 1: the strip is the whole row, no halo columns, one bulk copy per chunk (FR)
    uint32_t l2pf;       // n > 0: before griddepcontrol.wait, prefetch the band's first n chunks into L2
};

// s at offset `off` (site units) from ring0; off may reach into the mirror rows (< 0)
template <int FMT>
__device__ __forceinline__ int ring_get(const uint8_t* ring0, int off)
{
    if (FMT == kFmtU8) return ring0[off];
    return (ring0[off >> 3] >> (off & 7)) & 1;
}

// Without mirror rows a read above ring row 0 lands at the end of the ring: `wrap` = ring size in
// site units is added to a negative offset.
template <int FMT>
__device__ __forceinline__ int ring_getw(const uint8_t* ring0, int off, int wrap)
{
    return ring_get<FMT>(ring0, off + ((off >> 31) & wrap));
}

// Level 1 (a3, a4): draw, neighbour compare.  Returns true if the site goes on to level 2.
// Offset of the neighbour y of the site at soff.  FR ("full row": the strip is the whole lattice
// row, staged without halo columns, rows contiguous in shared memory): a horizontal step stays
// inside the row, colmask = row length in site units - 1 (a power of two minus one).
template <bool FR>
__device__ __forceinline__ int ring_nbr(int soff, uint32_t dir, int e, int colmask)
{
    if (!FR) return soff + e;
    const int m = dir >= 2u ? colmask : -1;
    return (soff & ~m) | ((soff + e) & m);
}

template <int FMT, bool FR = false>
__device__ __forceinline__ bool ring_level1(uint2 e, const uint8_t* ring0, const int* __restrict__ eoff,
                                            const StepKey& sk, uint4& out, int wrap, int colmask = 0)
{
    uint32_t x0, u;
    step_draw(sk, e.y, x0, u);
    const uint32_t dir = x0 >> 30;  // 0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1)
    const int soff = (int)e.x;
    const int sx = ring_get<FMT>(ring0, soff);
    const int sy = ring_getw<FMT>(ring0, ring_nbr<FR>(soff, dir, eoff[dir], colmask), wrap);  // wrap == 0 with mirror rows
    out = make_uint4(e.x | (dir << 30) | ((uint32_t)sx << 29), e.y, u, 0u);
    return sx != sy;
}

// Level 2 (a5-a7): payoff difference, acceptance, write.  Returns the change of the cooperator count.
template <int FMT, bool WRAP>
__device__ __forceinline__ int ring_stencil(int soff, uint32_t dir, int sx, const uint8_t* ring0,
                                            const int* __restrict__ eoff, int wrap)
{
    // e = step towards y, f = perpendicular step (site units)
    const int e = eoff[dir], f = eoff[4 + dir], f2 = 2 * f;
    const int pm1 = soff - e, pm2 = pm1 - e, p1 = soff + e, p2 = p1 + e, p3 = p2 + e;
    auto G = [&](int off) { return WRAP ? ring_getw<FMT>(ring0, off, wrap) : ring_get<FMT>(ring0, off); };
    // A_x - A_y with A = 5 s + 2 (nearest + diagonal) + axial distance-2 (include/pgg.h):
    // weights of x's 13-site stencil minus those of y's, y = x + e; s_x - s_y = 2 s_x - 1
    return G(pm2) + G(pm1) - G(p2) - G(p3) + 3 * (2 * sx - 1)
         + 2 * (G(pm1 + f) + G(pm1 - f) - G(p2 + f) - G(p2 - f))
         + G(soff + f2) + G(soff - f2) - G(p1 + f2) - G(p1 - f2);
}

// The stencil of a site near an end of its row in FR mode (and/or in ring row 0): row and column
// parts of every offset are formed separately, the column part wraps inside the row.
template <int FMT>
__device__ __forceinline__ int ring_stencil_fr(int soff, uint32_t dir, int sx, const uint8_t* ring0, int wrap,
                                               int colmask)
{
    const int col = soff & colmask, rowbase = soff - col, ps = colmask + 1;
    const int er = dir == 0u ? -1 : dir == 1u ? 1 : 0, ec = dir == 2u ? -1 : dir == 3u ? 1 : 0;
    const int fr = dir < 2u ? 0 : 1, fc = dir < 2u ? 1 : 0;
    auto S = [&](int a, int b) {
        int o = rowbase + (a * er + b * fr) * ps + ((col + a * ec + b * fc) & colmask);
        o += (o >> 31) & wrap;
        return ring_get<FMT>(ring0, o);
    };
    return S(-2, 0) + S(-1, 0) - S(2, 0) - S(3, 0) + 3 * (2 * sx - 1)
         + 2 * (S(-1, 1) + S(-1, -1) - S(2, 1) - S(2, -1))
         + S(0, 2) + S(0, -2) - S(1, 2) - S(1, -2);
}

// `wrap_below`: sites with soff below it (ring row 0) take the wrapping stencil; 0 with mirror rows.
template <int FMT, bool FR = false>
__device__ __forceinline__ int ring_accept(int soff, uint32_t dir, int sx, uint32_t site, uint32_t u,
                                           const uint8_t* ring0, const int* __restrict__ eoff,
                                           uint8_t* __restrict__ lat, const uint32_t* __restrict__ tbl,
                                           int wrap, int wrap_below, int colmask = 0)
{
    int dA;
    if (FR) {
        const int col = soff & colmask;
        dA = (soff < wrap_below || col < 3 || col > colmask - 3)
                 ? ring_stencil_fr<FMT>(soff, dir, sx, ring0, wrap, colmask)
                 : ring_stencil<FMT, false>(soff, dir, sx, ring0, eoff, 0);
    } else {
        dA = soff < wrap_below ? ring_stencil<FMT, true>(soff, dir, sx, ring0, eoff, wrap)
                               : ring_stencil<FMT, false>(soff, dir, sx, ring0, eoff, 0);
    }
    // table_index(dA, ds) = (ds + 1) * 51 + dA + 25 with ds = 2 s_x - 1
    if (u < tbl[sx * 102 + dA + 25]) {
        if (FMT == kFmtU8)
            lat[site] = (uint8_t)(1 - sx);
        else
            atomicXor(reinterpret_cast<uint32_t*>(lat) + (site >> 5), 1u << (site & 31u));
        return 1 - 2 * sx;
    }
    return 0;
}

// Level 2 on a Q2 entry (soff | dir << 30 | s_x << 29, site, u)
template <int FMT, bool FR = false>
__device__ __forceinline__ int ring_level2(uint4 w, const uint8_t* ring0, const int* __restrict__ eoff,
                                           uint8_t* __restrict__ lat, const uint32_t* __restrict__ tbl,
                                           int wrap, int wrap_below, int colmask = 0)
{
    return ring_accept<FMT, FR>((int)(w.x & 0x1FFFFFFFu), w.x >> 30, (int)((w.x >> 29) & 1u), w.y, w.z, ring0,
                                eoff, lat, tbl, wrap, wrap_below, colmask);
}

// Levels 1 and 2 of one queued site without the Q2 entry in between (the inline path)
struct RingDraw {
    uint32_t dir, u;
    int sx;
    bool go;
};
template <int FMT, bool FR = false>
__device__ __forceinline__ RingDraw ring_draw(uint2 e, const uint8_t* ring0, const int* __restrict__ eoff,
                                              const StepKey& sk, int wrap, int colmask = 0)
{
    RingDraw d;
    uint32_t x0;
    step_draw(sk, e.y, x0, d.u);
    d.dir = x0 >> 30;
    d.sx = ring_get<FMT>(ring0, (int)e.x);
    d.go = d.sx != ring_getw<FMT>(ring0, ring_nbr<FR>((int)e.x, d.dir, eoff[d.dir], colmask), wrap);
    return d;
}

// FULL: every strip is W bytes wide and every warp has an active row in every step (no ragged
// edges: the per-lane and per-step guards of the scan drop out).
// FR ("full row", implies FULL): one strip = the whole lattice row, staged without halo columns,
// so the rows of a chunk are contiguous in global AND shared memory and arrive as ONE bulk copy
// (rows of 512 B ... 8 KB copied singly stream at a fraction of the rate, profiles/
// DESIGN.md appendix A); the periodic column wrap is resolved in the few sites near a row end.
template <int FMT, bool FULL, bool FR>
__global__ void __launch_bounds__(kRingThreads, 1)
phase_ring_kernel(PhaseArgs a, uint32_t m, uint32_t k, RingPlan g)
{
    constexpr int kHalo = FR ? 0 : kRingHaloB;
    extern __shared__ __align__(128) uint8_t smem_raw[];
    const uint32_t NS = g.NS;
    const int RC = (int)g.RC, pitch = (int)g.pitch;
    const bool use_mirror = g.mirror != 0;
    uint8_t* ring0 = smem_raw + (use_mirror ? 3 * pitch : 0);  // three mirror rows in front of slot 0
    uint8_t* qbase = ring0 + (size_t)NS * g.slot_bytes;
    uint32_t* tbl = reinterpret_cast<uint32_t*>(qbase + kRingConsumers * RingCfg<FMT>::warp_q_bytes);
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(tbl + 160);  // full[NS], empty[NS]
    int* eoff = reinterpret_cast<int*>(bars + 2 * kRingMaxSlots);                 // e[4], f[4]
    __shared__ int delta_cta;

    const uint32_t b = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t L = a.L;
    uint8_t* lat = a.lats + (size_t)b * a.lat_bytes;
    const uint32_t bar_full = smem_u32(bars), bar_empty = bar_full + 8u * NS;

    // Programmatic dependent launch: the next phase's CTAs may take an SM as soon as this
    // kernel's CTA there has exited, and set themselves up; they touch nothing a previous
    // kernel wrote (the lattice, the phase order) before griddepcontrol.wait returns, i.e.
    // before the whole previous grid has completed and its writes are visible.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    for (int q = threadIdx.x; q < kTableSize; q += kRingThreads)
        tbl[q] = a.tables[(size_t)b * kTableSize + q];
    if (threadIdx.x == 0) {
        delta_cta = 0;
        for (uint32_t s = 0; s < NS; ++s) {
            mbar_init(bar_full + 8u * s, 1);
            mbar_init(bar_empty + 8u * s, kRingConsumers);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        const int ps = (FMT == kFmtU8) ? pitch : 8 * pitch;  // one row down, in site units
        eoff[0] = -ps; eoff[1] = ps; eoff[2] = -1; eoff[3] = 1;
        eoff[4] = 1;   eoff[5] = 1;  eoff[6] = ps; eoff[7] = ps;
    }
    if (g.l2pf && warp == kRingConsumers) {
        // L2PF: the first rows this CTA will stage, whatever the phase class turns out to be (the
        // class only shifts them by 0..3 rows).  A prefetch moves DRAM -> L2 only; L2 is the point
        // of coherence, so rows the previous phase is still writing cannot go stale.
        const uint32_t strip_ = blockIdx.x / g.nb, band_ = blockIdx.x - strip_ * g.nb;
        const long long S0_ = (long long)(((unsigned long long)band_ * g.n_super) / g.nb);
        const int j0_ = (int)(strip_ * g.W), wb_ = min((int)g.W, (int)g.row_bytes - j0_);
        const long long first = (long long)RC * (S0_ - 1) + RC - 3;
        const int n_rows = ((int)g.l2pf - 1) * RC + 3 + 4;  // the tail of chunk 0 and l2pf - 1 whole chunks, + 4 for the class
        for (int q = lane; q < n_rows; q += 32) {
            long long gi = (first + q) % (long long)L;
            if (gi < 0) gi += L;
            const uint8_t* src = lat + (size_t)gi * (size_t)g.row_bytes + j0_;
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"((uint32_t)wb_) : "memory");
        }
    }
    __syncthreads();
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const uint32_t cls = a.order[((size_t)b * a.order_stride + (m % a.order_stride)) * 16 + k];
    const int ci = (int)(cls >> 2), cj = (int)(cls & 3u);

    const uint32_t strip = blockIdx.x / g.nb, band = blockIdx.x - strip * g.nb;
    const uint32_t S0 = (uint32_t)(((unsigned long long)band * g.n_super) / g.nb);
    const uint32_t S1 = (uint32_t)(((unsigned long long)(band + 1) * g.n_super) / g.nb);
    const uint32_t n_steps = S1 - S0;
    const int j0b = (int)(strip * g.W);
    const int wb = min((int)g.W, (int)g.row_bytes - j0b);  // core bytes per row of this strip

    if (warp == kRingConsumers) {
        // ---------------- producer warp ----------------
        const int rb = (int)g.row_bytes;
        const bool left_edge = j0b == 0, right_edge = j0b + wb == rb;
        const uint32_t ring_s = smem_u32(ring0);
        const uint32_t n_chunks = n_steps ? n_steps + 1 : 0;
        const uint32_t row_tx = (uint32_t)(wb + 2 * kHalo);
        // first lattice row of chunk kc: the first active row of step S0 + kc - 1 (mod L)
        int row0 = (int)(((long long)RC * ((long long)S0 - 1) + ci) % (long long)L);
        if (row0 < 0) row0 += (int)L;
        uint32_t slot = 0, use = 0;  // chunk kc lives in slot kc % NS, use = kc / NS
        for (uint32_t kc = 0; kc < n_chunks; ++kc) {
            if (use > 0) mbar_wait(bar_empty + 8u * slot, (use - 1u) & 1u);
            const uint32_t bar = bar_full + 8u * slot;
            const int r_lo = kc == 0 ? RC - 3 : 0;  // of the prologue chunk only the tail is read
            const bool mirror = use_mirror && slot == NS - 1;     // its last three rows are also staged above slot 0
            if (lane == 0) mbar_expect_tx(bar, (uint32_t)(RC - r_lo + (mirror ? 3 : 0)) * row_tx);
            __syncwarp();
            if (FR) {
                // rows r_lo .. RC-1 of the chunk are contiguous in the lattice unless they cross its end
                const int g0 = (int)((uint32_t)(row0 + r_lo) % L), n = RC - r_lo;
                const int n1st = min(n, (int)L - g0);
                const uint32_t dst = ring_s + (slot * (uint32_t)RC + (uint32_t)r_lo) * (uint32_t)pitch;
                if (lane == 0) {
                    bulk_g2s(dst, lat + (size_t)g0 * (size_t)rb, (uint32_t)(n1st * rb), bar);
                    if (n1st < n) bulk_g2s(dst + (uint32_t)(n1st * rb), lat, (uint32_t)((n - n1st) * rb), bar);
                }
            } else
            for (int q = r_lo + lane; q < RC + (mirror ? 3 : 0); q += 32) {
                const int rr = q < RC ? q : q - 3;  // q >= RC: rows RC-3 .. RC-1 once more
                const int gi = (int)((uint32_t)(row0 + rr) % L);
                const uint8_t* src = lat + (size_t)gi * (size_t)rb;
                const uint32_t dst = q < RC ? ring_s + (slot * (uint32_t)RC + (uint32_t)rr) * (uint32_t)pitch
                                            : ring_s - (uint32_t)((RC + 3 - q) * pitch);
                if (!left_edge && !right_edge) {
                    bulk_g2s(dst, src + j0b - kRingHaloB, row_tx, bar);
                } else if (left_edge && !right_edge) {
                    bulk_g2s(dst, src + rb - kRingHaloB, kRingHaloB, bar);
                    bulk_g2s(dst + kRingHaloB, src, (uint32_t)(wb + kRingHaloB), bar);
                } else if (!left_edge && right_edge) {
                    bulk_g2s(dst, src + j0b - kRingHaloB, (uint32_t)(wb + kRingHaloB), bar);
                    bulk_g2s(dst + kRingHaloB + (uint32_t)wb, src, kRingHaloB, bar);
                } else {
                    bulk_g2s(dst, src + rb - kRingHaloB, kRingHaloB, bar);
                    bulk_g2s(dst + kRingHaloB, src, (uint32_t)wb, bar);
                    bulk_g2s(dst + kRingHaloB + (uint32_t)wb, src, kRingHaloB, bar);
                }
            }
            row0 += RC;
            if (row0 >= (int)L) row0 %= (int)L;
            if (++slot == NS) { slot = 0; ++use; }
        }
    } else {
        // ---------------- consumer warps ----------------
        const StepKey sk = make_step_key(a.seeds[b], a.t_begin + m, k, cls);
        uint2* q1 = reinterpret_cast<uint2*>(qbase + warp * RingCfg<FMT>::warp_q_bytes);
        uint4* q2 = reinterpret_cast<uint4*>(q1 + kRingQ1Cap);
        const uint32_t lt = (1u << lane) - 1u;
        const int rho = warp >> g.tpr_log2, tau = warp & ((1 << g.tpr_log2) - 1);
        const int colb = tau * kRingTaskB + 16 * lane;  // first core byte of this lane's 16
        const bool in = colb < wb;
        const bool rotate = FULL && FMT == kFmtU8 && g.tpr_log2 == 4 && g.rotate != 0;
        const int slot_bytes = (int)g.slot_bytes;
        const int ring_bytes = (int)NS * slot_bytes;
        // site units; both 0 with mirror rows (then no read ever wraps)
        const int ps_sites = (FMT == kFmtU8) ? pitch : 8 * pitch;
        const int wrap = use_mirror ? 0 : ((FMT == kFmtU8) ? ring_bytes : 8 * ring_bytes);
        const int wrap_below = use_mirror ? 0 : ps_sites;
        const int colmask = FR ? ps_sites - 1 : 0;  // FR: pitch = row length, a power of two
        // Q1 is linear, entries [0, n1); Q2 is a ring of kRingQ2Cap entries, [h2, h2 + n2).
        // o1 / o2 = how many entries at the front were queued by the previous step (they
        // must be finished before this step ends, when their rows are released).
        uint32_t n1 = 0, n2 = 0, h2 = 0, o1 = 0, o2 = 0;
        int delta = 0;
        uint32_t slot = 1 % NS;                // of chunk s + 1
        uint32_t par = (1 / NS) & 1u;          // parity of its "full" barrier
        uint32_t rel_slot = 0;                 // slot of chunk s - 1
        // this lane's 16 bytes of the warp's active row: byte offset from ring0, and the
        // lattice site index of the first of them
        int rowoff = (int)slot * slot_bytes + 4 * rho * pitch + kHalo + colb;
        // byte offset from this lane's 16 bytes to the same columns one lattice row up
        const int up_wrapped = (use_mirror || rho != 0) ? -pitch : ring_bytes - pitch;
        int upoff = (slot == 0) ? up_wrapped : -pitch;
        uint32_t site0 = (uint32_t)(RC * (int)S0 + 4 * rho + ci) * L
                       + (uint32_t)((FMT == kFmtU8) ? j0b + colb : 8 * (j0b + colb));
        const uint32_t site_step = (uint32_t)RC * L;
        // steps in which this warp's active row exists (the last step of a strip may be ragged)
        const uint32_t first_group = S0 * g.R + (uint32_t)rho;
        const uint32_t n_act = first_group >= g.n_groups ? 0u
                             : min(n_steps, (g.n_groups - first_group + g.R - 1) / g.R);

        // level 2 on the first `cnt` (<= 32) entries of Q2
        auto run_level2 = [&](uint32_t cnt) {
            if ((uint32_t)lane < cnt)
                delta += ring_level2<FMT, FR>(q2[(h2 + lane) & (kRingQ2Cap - 1)], ring0, eoff, lat, tbl, wrap, wrap_below, colmask);
            __syncwarp();  // entries are read before a later append may overwrite them
            h2 += cnt;
            n2 -= cnt;
            o2 = o2 > cnt ? o2 - cnt : 0u;
        };
        // Q2 append of one level-1 batch whose first `n_old` lanes hold old entries
        auto push2 = [&](bool go, const uint4& w, uint32_t n_old) {
            if (!RingCfg<FMT>::q2) {
                if (go) delta += ring_level2<FMT, FR>(w, ring0, eoff, lat, tbl, wrap, wrap_below, colmask);
                return;
            }
            const uint32_t mk = __ballot_sync(0xFFFFFFFFu, go);
            if (go) q2[(h2 + n2 + __popc(mk & lt)) & (kRingQ2Cap - 1)] = w;
            if (n_old) {
                const uint32_t c = __popc(mk & ((1u << n_old) - 1u));  // n_old < 32
                if (c) o2 = n2 + c;
            }
            n2 += __popc(mk);
            __syncwarp();
            if (n2 >= 32u) run_level2(32u);
        };
        // level 1 on `cnt` (<= 32) entries of Q1 starting at `head`
        auto run_level1 = [&](uint32_t head, uint32_t cnt, uint32_t n_old) {
            if (!RingCfg<FMT>::q2) {
                if ((uint32_t)lane < cnt) {
                    const uint2 e = q1[head + lane];
                    const RingDraw d = ring_draw<FMT, FR>(e, ring0, eoff, sk, wrap, colmask);
                    if (d.go)
                        delta += ring_accept<FMT, FR>((int)e.x, d.dir, d.sx, e.y, d.u, ring0, eoff, lat, tbl, wrap, wrap_below, colmask);
                }
                return;
            }
            uint4 w;
            bool go = false;
            if ((uint32_t)lane < cnt) go = ring_level1<FMT, FR>(q1[head + lane], ring0, eoff, sk, w, wrap, colmask);
            push2(go, w, n_old);
        };
        // full batches from the front of Q1 (two at a time while 64 wait); the leftover
        // (< 32) moves to the front.  Old entries (o1 < 32 of them) are in the first batch.
        auto run_batches = [&]() {
            if (n1 < 32u) return;
            uint32_t head = 0;
            if (n1 >= 64u) {
                do {
                    if (!RingCfg<FMT>::q2) {  // two independent Philox chains, then the two stencils
                        const uint2 ea = q1[head + lane], eb = q1[head + 32 + lane];
                        const RingDraw da = ring_draw<FMT, FR>(ea, ring0, eoff, sk, wrap, colmask);
                        const RingDraw db = ring_draw<FMT, FR>(eb, ring0, eoff, sk, wrap, colmask);
                        if (da.go)
                            delta += ring_accept<FMT, FR>((int)ea.x, da.dir, da.sx, ea.y, da.u, ring0, eoff, lat, tbl, wrap, wrap_below, colmask);
                        if (db.go)
                            delta += ring_accept<FMT, FR>((int)eb.x, db.dir, db.sx, eb.y, db.u, ring0, eoff, lat, tbl, wrap, wrap_below, colmask);
                        head += 64u;
                        continue;
                    }
                    uint4 wa, wb2;
                    const bool ga = ring_level1<FMT, FR>(q1[head + lane], ring0, eoff, sk, wa, wrap, colmask);
                    const bool gb = ring_level1<FMT, FR>(q1[head + 32 + lane], ring0, eoff, sk, wb2, wrap, colmask);
                    push2(ga, wa, head ? 0u : o1);
                    push2(gb, wb2, 0u);
                    head += 64u;
                } while (n1 - head >= 64u);
                if (n1 - head >= 32u) {
                    run_level1(head, 32u, 0u);
                    head += 32u;
                }
            } else {
                run_level1(0u, 32u, o1);
                head = 32u;
            }
            const uint32_t left = n1 - head;
            uint2 e = make_uint2(0u, 0u);
            if ((uint32_t)lane < left) e = q1[head + lane];
            __syncwarp();
            if ((uint32_t)lane < left) q1[lane] = e;
            __syncwarp();
            n1 = left;
            o1 = 0;
        };

        if (n_steps) mbar_wait(bar_full, 0u);
        for (uint32_t s = 0; s < n_steps; ++s) {
            mbar_wait(bar_full + 8u * slot, par);
            // ROTATE: warp w takes column task (w + s) mod 16 of step s, so that no warp is tied to
            // the busiest columns of the band for good (queue entries are self-contained)
            const int rot = rotate ? ((((warp + (int)s) & 15) - tau) * kRingTaskB) : 0;
            if (FULL || s < n_act) {
                const uint8_t* rowp = ring0 + rowoff + rot;
                uint4 wc = make_uint4(0, 0, 0, 0), wu = wc, wd = wc;
                uint32_t pv = 0, nx = 0;
                if (FULL || in) {
                    wc = *reinterpret_cast<const uint4*>(rowp);
                    wu = *reinterpret_cast<const uint4*>(rowp + upoff);
                    wd = *reinterpret_cast<const uint4*>(rowp + pitch);
                    // FR: the word left of the row's first / right of its last is the row's other end
                    pv = *reinterpret_cast<const uint32_t*>(rowp - 4 + ((FR && colb + rot == 0) ? pitch : 0));
                    nx = *reinterpret_cast<const uint32_t*>(rowp + 16 - ((FR && colb + rot + 16 == pitch) ? pitch : 0));
                }
                const uint32_t c4[4] = {wc.x, wc.y, wc.z, wc.w};
                const uint32_t u4[4] = {wu.x, wu.y, wu.z, wu.w};
                const uint32_t d4[4] = {wd.x, wd.y, wd.z, wd.w};
                uint32_t nb[4];
                if (FMT == kFmtU8) {
                    // word w = sites 4w..4w+3 of this lane's 16; the active one is byte cj
                    const uint32_t bm = 0xFFu << (8 * cj);
#pragma unroll
                    for (int w = 0; w < 4; ++w) {
                        const uint32_t lw = __funnelshift_l(w == 0 ? pv : c4[w - 1], c4[w], 8);
                        const uint32_t rw = __funnelshift_r(c4[w], w == 3 ? nx : c4[w + 1], 8);
                        nb[w] = ((c4[w] ^ u4[w]) | (c4[w] ^ d4[w]) | (c4[w] ^ lw) | (c4[w] ^ rw)) & bm;  // S9
                    }
                    if (__any_sync(0xFFFFFFFFu, (nb[0] | nb[1] | nb[2] | nb[3]) != 0u)) {
                        const uint32_t so = (uint32_t)(rowoff + rot + cj), si = site0 + (uint32_t)(rot + cj);
#pragma unroll
                        for (int w = 0; w < 4; ++w) {
                            const bool pred = nb[w] != 0u;
                            const uint32_t mk = __ballot_sync(0xFFFFFFFFu, pred);
                            if (pred) q1[n1 + __popc(mk & lt)] = make_uint2(so + 4u * w, si + 4u * w);
                            n1 += __popc(mk);
                        }
                        __syncwarp();
                        run_batches();
                    }
                } else {
                    // word w = 32 sites; the 8 active ones are bits cj + 4 b
                    const uint32_t cm = 0x11111111u << cj;
#pragma unroll
                    for (int w = 0; w < 4; ++w) {
                        const uint32_t lw = __funnelshift_l(w == 0 ? pv : c4[w - 1], c4[w], 1);
                        const uint32_t rw = __funnelshift_r(c4[w], w == 3 ? nx : c4[w + 1], 1);
                        nb[w] = ((c4[w] ^ u4[w]) | (c4[w] ^ d4[w]) | (c4[w] ^ lw) | (c4[w] ^ rw)) & cm;  // S9
                    }
#pragma unroll
                    for (int w = 0; w < 4; ++w) {
                        if (__any_sync(0xFFFFFFFFu, nb[w] != 0u)) {
                            const uint32_t so = (uint32_t)(8 * rowoff + 32 * w + cj);
                            const uint32_t si = site0 + (uint32_t)(32 * w + cj);
#pragma unroll
                            for (int bb = 0; bb < 8; ++bb) {
                                const bool pred = (nb[w] >> (cj + 4 * bb)) & 1u;
                                const uint32_t mk = __ballot_sync(0xFFFFFFFFu, pred);
                                if (pred) q1[n1 + __popc(mk & lt)] = make_uint2(so + 4u * bb, si + 4u * bb);
                                n1 += __popc(mk);
                                if ((bb & 3) == 3) {  // at most 31 + 4 * 32 entries: fits kRingQ1Cap
                                    __syncwarp();
                                    run_batches();
                                }
                            }
                        }
                    }
                }
            }
            // sites queued by step s-1 must be finished now: their rows are about to be released
            if (o1) {  // then n1 < 32
                run_level1(0u, n1, o1);
                n1 = 0;
            }
            if (RingCfg<FMT>::q2 && o2) run_level2(n2);  // then n2 < 32
            if (s > 0) {
                if (lane == 0) mbar_arrive(bar_empty + 8u * rel_slot);  // chunk s-1 is free
                if (++rel_slot == NS) rel_slot = 0;
            }
            o1 = n1;
            o2 = n2;
            site0 += site_step;
            rowoff += slot_bytes;
            upoff = -pitch;
            if (++slot == NS) { slot = 0; par ^= 1u; rowoff -= ring_bytes; upoff = up_wrapped; }
        }
        // drain: everything left was queued by the last step
        if (n1) {
            run_level1(0u, n1, 0u);
            n1 = 0;
        }
        if (n2) run_level2(n2);
        if (a.deltas != nullptr) {
            delta = __reduce_add_sync(0xFFFFFFFFu, delta);
            if (lane == 0 && delta != 0) atomicAdd(&delta_cta, delta);
        }
    }
    __syncthreads();
    if (a.deltas != nullptr && threadIdx.x == 0 && delta_cta != 0)
        atomicAdd(a.deltas + (size_t)b * a.n_mcs + m, (unsigned long long)(long long)delta_cta);
}

// ---------------------------------------------------------------------------
// Host side
// ---------------------------------------------------------------------------
inline bool ring_supported(int fmt, uint32_t L)
{
    if (L >= 65536) return false;
    return fmt == kFmtU8 ? (L % 16 == 0) : (L % 128 == 0);  // rows are multiples of 16 bytes
}

inline int ring_plan(int fmt, uint32_t L, uint32_t B, RingPlan* p, bool allow_fullrow = true)
{
    int sm_count = 0, smem_optin = 0;  // per call: the function attribute is per device, and a plan costs nothing next to 16 n_mcs launches
    {
        int dev = 0, sms = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return (int)e;
        const void* kernels[6] = {
            (const void*)phase_ring_kernel<kFmtU8, false, false>, (const void*)phase_ring_kernel<kFmtU8, true, false>,
            (const void*)phase_ring_kernel<kFmtU8, true, true>, (const void*)phase_ring_kernel<kFmtBits, false, false>,
            (const void*)phase_ring_kernel<kFmtBits, true, false>, (const void*)phase_ring_kernel<kFmtBits, true, true>};
        for (const void* kern : kernels) {
            e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 256);
            if (e != cudaSuccess) return (int)e;
        }
        sm_count = sms;
    }
    p->row_bytes = fmt == kFmtU8 ? L : L / 8;
    const uint32_t tasks = (p->row_bytes + kRingTaskB - 1) / kRingTaskB;
    uint32_t tpr_max = 4;
    if (const char* e = getenv("PGG_RING_TPR_LOG2")) tpr_max = (uint32_t)atoi(e);
    if (tpr_max > 4) tpr_max = 4;
    uint32_t tpr_log2 = 0;
    while ((1u << tpr_log2) < tasks && tpr_log2 < tpr_max) ++tpr_log2;
    p->tpr_log2 = tpr_log2;
    p->W = (1u << tpr_log2) * kRingTaskB;
    p->n_strips = (p->row_bytes + p->W - 1) / p->W;
    p->R = kRingConsumers >> tpr_log2;
    p->RC = 4 * p->R;
    // measured: a 2x gain for uint8 (16 x 2048^2: 31.7 -> 14.6 us per launch), a loss for the
    // bit-packed layout (L = 16384: 64 -> 88 us), so bit-packed takes it only on request
    const bool fr_ok = allow_fullrow && p->n_strips == 1 && p->W == p->row_bytes;
    p->fullrow = (fr_ok && fmt == kFmtU8) ? 1u : 0u;
    if (const char* e = getenv("PGG_RING_FULLROW")) p->fullrow = (fr_ok && atoi(e)) ? 1u : 0u;
    p->pitch = p->fullrow ? p->W : p->W + 2 * kRingHaloB;
    p->slot_bytes = p->RC * p->pitch;
    p->n_groups = L / 4;
    p->n_super = (p->n_groups + p->R - 1) / p->R;
    uint32_t per_strip = (uint32_t)sm_count / (p->n_strips * B);
    if (per_strip < 1) per_strip = 1;
    p->nb = p->n_super < per_strip ? p->n_super : per_strip;
    const uint32_t max_chunks = (p->n_super + p->nb - 1) / p->nb + 1;
    uint32_t want = kRingMaxSlots;
    if (const char* e = getenv("PGG_RING_SLOTS")) want = (uint32_t)atoi(e);
    if (want > (uint32_t)kRingMaxSlots) want = kRingMaxSlots;
    if (want < 3) want = 3;
    p->mirror = 0;
    if (const char* e = getenv("PGG_RING_MIRROR")) p->mirror = (atoi(e) && !p->fullrow) ? 1u : 0u;
    p->rotate = 1;
    if (const char* e = getenv("PGG_RING_ROTATE")) p->rotate = atoi(e) ? 1u : 0u;
    p->l2pf = 3;  // chunks; measured: 58.6 -> 58.1 us per launch (DESIGN.md appendix A)
    if (const char* e = getenv("PGG_RING_L2PF")) p->l2pf = (uint32_t)std::max(0, std::min(64, atoi(e)));
    const uint32_t fixed = (uint32_t)(fmt == kFmtU8 ? RingCfg<kFmtU8>::fixed_bytes : RingCfg<kFmtBits>::fixed_bytes)
                         + (p->mirror ? 3 * p->pitch : 0);
    while (want > 3 && want * p->slot_bytes + fixed > (uint32_t)smem_optin - 256) --want;
    if (max_chunks < want) want = max_chunks < 3 ? 3 : max_chunks;
    p->NS = want;
    p->smem_bytes = p->NS * p->slot_bytes + fixed;
    return 0;
}

inline void ring_launch(const RingPlan& p, int fmt, const PhaseArgs& a, uint32_t m, uint32_t k,
                        uint32_t B, cudaStream_t stream)
{
    static const bool pdl = [] { const char* e = getenv("PGG_PDL"); return e == nullptr || atoi(e) != 0; }();
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(p.n_strips * p.nb, B);
    cfg.blockDim = dim3(kRingThreads);
    cfg.dynamicSmemBytes = p.smem_bytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const bool full = p.row_bytes % p.W == 0 && p.n_groups % p.R == 0;
    if (fmt == kFmtU8) {
        if (p.fullrow) cudaLaunchKernelEx(&cfg, phase_ring_kernel<kFmtU8, true, true>, a, m, k, p);
        else if (full) cudaLaunchKernelEx(&cfg, phase_ring_kernel<kFmtU8, true, false>, a, m, k, p);
        else cudaLaunchKernelEx(&cfg, phase_ring_kernel<kFmtU8, false, false>, a, m, k, p);
    } else {
        if (p.fullrow) cudaLaunchKernelEx(&cfg, phase_ring_kernel<kFmtBits, true, true>, a, m, k, p);
        else if (full) cudaLaunchKernelEx(&cfg, phase_ring_kernel<kFmtBits, true, false>, a, m, k, p);
        else cudaLaunchKernelEx(&cfg, phase_ring_kernel<kFmtBits, false, false>, a, m, k, p);
    }
}

}  // namespace pgg
