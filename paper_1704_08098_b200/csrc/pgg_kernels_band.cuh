// pgg_kernels_band.cuh -- the BAND phase kernel (K1 uint8, K2 bit-packed).
//
// Measured on B200 (DESIGN.md appendix A): cp.async.bulk copies
// of ~0.5 KB issued by one warp deliver only ~2.2 TB/s chip-wide, copies of
// >= 1 KB reach 5.6-5.8 TB/s.  So the lattice is not cut into square tiles
// (short rows, 16 % halo re-reads) but into column STRIPS of up to 8 KB, and
// every persistent CTA streams one BAND of consecutive lattice rows of a strip
// through a ring of row chunks in shared memory: each lattice row is fetched
// exactly once per phase by one large bulk-async copy (SASS UBLKCP, completing
// on an mbarrier), plus 16 bytes of column halo on each side (3 sites are
// needed; 16 bytes keep every copy 16-byte aligned; at the lattice edge the
// halo is the periodic image).
//
//   ring    = [slot 0][slot 1]...[slot NS-1], slot = RC rows of `pitch` bytes
//   chunk k = RC = 4 R consecutive lattice rows of the band, the first one an
//             active row (row % 4 == ci); lives in slot k % NS.
//   step s  = the R active rows of chunk s+1; their stencils reach 3 rows up
//             (tail of chunk s) and 3 rows down (inside chunk s+1).  When chunk
//             s+1 sits in slot 0 the rows above it are the tail of slot NS-1:
//             a negative row offset from ring row 0 gets `ring_bytes` added.
//
// 16 consumer warps + 1 producer warp.  Consumer warp w owns 128 active sites
// (uint8; 512 bytes) or 1024 (bit-packed) of active row w / tpr, column task
// w % tpr, of every step:
//   scan    S9 bulk test ("all four neighbours equal s_x": no draw can change
//           the site) on 16 bytes per lane with word-wide logic; survivors go
//           to the warp's queue Q1;
//   level 1 batches of 32 from Q1: Philox draw (a3), s_y (a4); sites with
//           s_y != s_x go to queue Q2 with their u;
//   level 2 batches of 32 from Q2: A_x - A_y (a5), threshold compare (a6),
//           in-place write (a7), cooperator-count delta (a8).
// Both queues are FIFO and keep leftovers (< 32) across ONE step boundary: a
// warp releases chunk s-1 at the end of step s, after every site queued in
// step s-1 has been finished.
#pragma once
#include "pgg_kernels_pipe.cuh"

namespace pgg {

constexpr int kBandConsumers = 16;
constexpr int kBandThreads = (kBandConsumers + 1) * 32;
constexpr int kBandTaskB = 512;     // bytes of one lattice row that one warp scans per step
constexpr int kBandHaloB = 16;
constexpr int kBandQ2Cap = 64;      // Q2 entries (8 bytes each) per warp
constexpr int kBandMaxSlots = 6;

// Q1 entries (4 bytes) per warp: leftover (< 32) + the sites one scan round can add
template <int FMT> struct BandQ1 { static constexpr int cap = (FMT == kFmtU8) ? 32 + 128 : 32 + 256; };

template <int FMT>
constexpr int band_fixed_bytes()
{
    return kBandConsumers * (BandQ1<FMT>::cap * 4 + kBandQ2Cap * 8) + 160 * 4 + 2 * kBandMaxSlots * 8 + 128;
}

struct BandPlan {
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
};

// Q1 entry: step parity << 31 | ring row << 16 | site column (core-relative).
// Q2 entry: .x = Q1 entry | dir << 29 | s_x << 28, .y = u.   (ring row < 2^12)
struct BandCtx {
    const uint8_t* ring0;  // slot 0, row 0
    int pitch;
    int ring_bytes;        // NS * slot_bytes
    int rc_mask;           // RC - 1
    int j0;                // first core SITE column of the strip
    uint32_t L;
};

// lattice site index of a queued entry
__device__ __forceinline__ uint32_t band_site(uint32_t e, uint32_t par_cur, int grow_cur, const BandCtx& cx)
{
    const int pos = (int)((e >> 16) & 0xFFFu), c = (int)(e & 0xFFFFu);
    const int gi = (((e >> 31) == par_cur) ? grow_cur : grow_cur - (cx.rc_mask + 1)) + (pos & cx.rc_mask);
    return (uint32_t)gi * cx.L + (uint32_t)(cx.j0 + c);
}

// One site of the staged ring: row `pos` + rr (rr in [-3, 3]), site column c + cc.
// `fix` = ring_bytes if pos == 0 (rows above ring row 0 are the tail of the last slot), else 0.
template <int FMT>
__device__ __forceinline__ int band_get(const uint8_t* rowp, int pitch, int c, int rr, int cc, int fixr)
{
    // fixr: 0, or `fix` when this access has rr < 0
    if (FMT == kFmtU8) return rowp[rr * pitch + c + cc + fixr];
    const int q = c + cc;
    return (rowp[rr * pitch + (q >> 3) + fixr] >> (q & 7)) & 1;
}

// Level 1 (a3, a4): draw, neighbour compare.  Returns true if the site goes on to level 2.
template <int FMT>
__device__ __forceinline__ bool band_level1(uint32_t e, uint32_t par_cur, int grow_cur, const BandCtx& cx,
                                            const StepKey& sk, uint2& out)
{
    const uint32_t site = band_site(e, par_cur, grow_cur, cx);
    uint32_t x0, u;
    step_draw(sk, site, x0, u);
    const uint32_t dir = x0 >> 30;  // 0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1)
    const int pos = (int)((e >> 16) & 0xFFFu);
    const int c = (int)(e & 0xFFFFu) + ((FMT == kFmtU8) ? kBandHaloB : 8 * kBandHaloB);
    const uint8_t* rowp = cx.ring0 + pos * cx.pitch;
    const int er = dir == 0 ? -1 : dir == 1 ? 1 : 0;
    const int ec = dir == 2 ? -1 : dir == 3 ? 1 : 0;
    const int fix = (pos == 0 && dir == 0) ? cx.ring_bytes : 0;
    const int sx = band_get<FMT>(rowp, cx.pitch, c, 0, 0, 0);
    const int sy = band_get<FMT>(rowp, cx.pitch, c, er, ec, fix);
    out.x = e | (dir << 29) | ((uint32_t)sx << 28);
    out.y = u;
    return sx != sy;
}

// Level 2 (a5-a7): payoff difference, acceptance, write.  Returns the change of the cooperator count.
template <int FMT>
__device__ __forceinline__ int band_level2(uint2 w, uint32_t par_cur, int grow_cur, const BandCtx& cx,
                                           uint8_t* __restrict__ lat, const uint32_t* __restrict__ tbl)
{
    const uint32_t e = w.x, u = w.y;
    const uint32_t dir = (e >> 29) & 3u;
    const int sx = (int)((e >> 28) & 1u), sy = 1 - sx;
    const int pos = (int)((e >> 16) & 0xFFFu);
    const int c = (int)(e & 0xFFFFu) + ((FMT == kFmtU8) ? kBandHaloB : 8 * kBandHaloB);
    const uint8_t* rowp = cx.ring0 + pos * cx.pitch;
    // e = unit step towards y, f = perpendicular unit step: (ring row, site column)
    const int er = dir == 0 ? -1 : dir == 1 ? 1 : 0;
    const int ec = dir == 2 ? -1 : dir == 3 ? 1 : 0;
    const int fr = dir < 2 ? 0 : 1, fc = dir < 2 ? 1 : 0;
    // accesses whose ring row is above row `pos`: a > 0 when dir == 0, a < 0 when dir == 1,
    // b < 0 when dir >= 2 (then, and only if pos == 0, they live at the end of the ring)
    const int fix = pos == 0 ? cx.ring_bytes : 0;
    const int fa_pos = dir == 0 ? fix : 0, fa_neg = dir == 1 ? fix : 0, fb_neg = dir >= 2 ? fix : 0;
    auto S = [&](int a, int b) {
        const int fixr = (a > 0 ? fa_pos : 0) + (a < 0 ? fa_neg : 0) + (b < 0 ? fb_neg : 0);
        return band_get<FMT>(rowp, cx.pitch, c, a * er + b * fr, a * ec + b * fc, fixr);
    };
    // A_x - A_y with A = 5 s + 2 (nearest + diagonal) + axial distance-2 (include/pgg.h):
    // weights of x's 13-site stencil minus those of y's, at offset (a along e, b along f)
    const int dA = S(-2, 0) + S(-1, 0) - S(2, 0) - S(3, 0) + 3 * (sx - sy)
                 + 2 * (S(-1, 1) + S(-1, -1) - S(2, 1) - S(2, -1))
                 + S(0, 2) + S(0, -2) - S(1, 2) - S(1, -2);
    if (u < tbl[table_index(dA, sx - sy)]) {
        const uint32_t site = band_site(e, par_cur, grow_cur, cx);
        if (FMT == kFmtU8)
            lat[site] = (uint8_t)sy;
        else
            atomicXor(reinterpret_cast<uint32_t*>(lat) + (site >> 5), 1u << (site & 31u));
        return sy - sx;
    }
    return 0;
}

template <int FMT>
__global__ void __launch_bounds__(kBandThreads, 1)
phase_band_kernel(PhaseArgs a, uint32_t m, uint32_t k, BandPlan g)
{
    extern __shared__ __align__(128) uint8_t smem_raw[];
    constexpr int kQ1 = BandQ1<FMT>::cap;
    const uint32_t NS = g.NS;
    uint8_t* ring0 = smem_raw;
    uint8_t* qbase = smem_raw + (size_t)NS * g.slot_bytes;
    uint32_t* tbl = reinterpret_cast<uint32_t*>(qbase + kBandConsumers * (kQ1 * 4 + kBandQ2Cap * 8));
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(tbl + 160);  // full[NS], empty[NS]
    __shared__ int delta_cta;

    const uint32_t b = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t L = a.L;
    uint8_t* lat = a.lats + (size_t)b * a.lat_bytes;
    const uint32_t bar_full = smem_u32(bars), bar_empty = bar_full + 8u * NS;

    // programmatic dependent launch, as in pgg_kernels_ring.cuh: set up while the previous
    // phase drains, touch the lattice and the phase order only after griddepcontrol.wait
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    for (int q = threadIdx.x; q < kTableSize; q += kBandThreads)
        tbl[q] = a.tables[(size_t)b * kTableSize + q];
    if (threadIdx.x == 0) {
        delta_cta = 0;
        for (uint32_t s = 0; s < NS; ++s) {
            mbar_init(bar_full + 8u * s, 1);
            mbar_init(bar_empty + 8u * s, kBandConsumers);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const uint32_t cls = a.order[((size_t)b * a.order_stride + (m % a.order_stride)) * 16 + k];
    const int ci = (int)(cls >> 2), cj = (int)(cls & 3u);

    const uint32_t strip = blockIdx.x / g.nb, band = blockIdx.x - strip * g.nb;
    const uint32_t S0 = (uint32_t)(((unsigned long long)band * g.n_super) / g.nb);
    const uint32_t S1 = (uint32_t)(((unsigned long long)(band + 1) * g.n_super) / g.nb);
    const uint32_t n_steps = S1 - S0;
    const int RC = (int)g.RC, pitch = (int)g.pitch;
    const int j0b = (int)(strip * g.W);
    const int wb = min((int)g.W, (int)g.row_bytes - j0b);  // core bytes per row of this strip

    if (warp == kBandConsumers) {
        // ---------------- producer warp ----------------
        const int rb = (int)g.row_bytes;
        const bool left_edge = j0b == 0, right_edge = j0b + wb == rb;
        const uint32_t ring_s = smem_u32(ring0);
        const uint32_t n_chunks = n_steps ? n_steps + 1 : 0;
        // first lattice row of chunk kc: the first active row of step S0 + kc - 1 (mod L)
        int row0 = (int)(((long long)RC * ((long long)S0 - 1) + ci) % (long long)L);
        if (row0 < 0) row0 += (int)L;
        uint32_t slot = 0, use = 0;  // chunk kc lives in slot kc % NS, use = kc / NS
        for (uint32_t kc = 0; kc < n_chunks; ++kc) {
            if (use > 0) mbar_wait(bar_empty + 8u * slot, (use - 1u) & 1u);
            const uint32_t bar = bar_full + 8u * slot;
            const int r_lo = kc == 0 ? RC - 3 : 0;  // of the prologue chunk only the tail is read
            if (lane == 0) mbar_expect_tx(bar, (uint32_t)((RC - r_lo) * (wb + 2 * kBandHaloB)));
            __syncwarp();
            for (int rr = r_lo + lane; rr < RC; rr += 32) {
                const int gi = (int)((uint32_t)(row0 + rr) % L);
                const uint8_t* src = lat + (size_t)gi * (size_t)rb;
                const uint32_t dst = ring_s + (slot * (uint32_t)RC + (uint32_t)rr) * (uint32_t)pitch;
                if (!left_edge && !right_edge) {
                    bulk_g2s(dst, src + j0b - kBandHaloB, (uint32_t)(wb + 2 * kBandHaloB), bar);
                } else if (left_edge && !right_edge) {
                    bulk_g2s(dst, src + rb - kBandHaloB, kBandHaloB, bar);
                    bulk_g2s(dst + kBandHaloB, src, (uint32_t)(wb + kBandHaloB), bar);
                } else if (!left_edge && right_edge) {
                    bulk_g2s(dst, src + j0b - kBandHaloB, (uint32_t)(wb + kBandHaloB), bar);
                    bulk_g2s(dst + kBandHaloB + (uint32_t)wb, src, kBandHaloB, bar);
                } else {
                    bulk_g2s(dst, src + rb - kBandHaloB, kBandHaloB, bar);
                    bulk_g2s(dst + kBandHaloB, src, (uint32_t)wb, bar);
                    bulk_g2s(dst + kBandHaloB + (uint32_t)wb, src, kBandHaloB, bar);
                }
            }
            row0 += RC;
            if (row0 >= (int)L) row0 %= (int)L;
            if (++slot == NS) { slot = 0; ++use; }
        }
    } else {
        // ---------------- consumer warps ----------------
        const StepKey sk = make_step_key(a.seeds[b], a.t_begin + m, k, cls);
        uint32_t* q1 = reinterpret_cast<uint32_t*>(qbase + warp * (kQ1 * 4 + kBandQ2Cap * 8));
        uint2* q2 = reinterpret_cast<uint2*>(q1 + kQ1);
        const uint32_t lt = (1u << lane) - 1u;
        const int rho = warp >> g.tpr_log2, tau = warp & ((1 << g.tpr_log2) - 1);
        const int colb = tau * kBandTaskB + 16 * lane;  // first core byte of this lane's 16
        const bool in = colb < wb;
        BandCtx cx;
        cx.ring0 = ring0;
        cx.pitch = pitch;
        cx.ring_bytes = (int)(NS * g.slot_bytes);
        cx.rc_mask = RC - 1;
        cx.j0 = (FMT == kFmtU8) ? j0b : j0b * 8;
        cx.L = L;
        // Both queues are linear, entries [0, n).  n1_old / n2_old = how many entries at the
        // front were queued by the previous step (they must be finished before this step ends).
        uint32_t n1 = 0, n2 = 0, n1_old = 0, n2_old = 0;
        int delta = 0;
        uint32_t slot = 1 % NS, use = 1 / NS;       // of chunk s + 1
        uint32_t rel_slot = 0;                      // slot of chunk s - 1
        uint32_t par = 0;
        int grow_cur = RC * (int)S0 + ci;           // lattice row of the step's first active row
        uint32_t group = S0 * g.R + (uint32_t)rho;  // index of this warp's active row among the class rows

        // level 2 on the first `cnt` (<= 32) entries of Q2; the rest moves to the front
        auto run_level2 = [&](uint32_t cnt) {
            uint2 w = make_uint2(0u, 0u), mv = w;
            if ((uint32_t)lane < cnt) w = q2[lane];
            const uint32_t left = n2 - cnt;
            if ((uint32_t)lane < left) mv = q2[cnt + lane];
            __syncwarp();
            if ((uint32_t)lane < left) q2[lane] = mv;
            if ((uint32_t)lane < cnt) delta += band_level2<FMT>(w, par, grow_cur, cx, lat, tbl);
            __syncwarp();
            n2 = left;
            n2_old = n2_old > cnt ? n2_old - cnt : 0u;
        };
        // level 1 on the first `cnt` (<= 32) entries of Q1 starting at `head`
        auto run_level1 = [&](uint32_t head, uint32_t cnt, bool has_old) {
            uint2 w;
            bool go = false;
            if ((uint32_t)lane < cnt) go = band_level1<FMT>(q1[head + lane], par, grow_cur, cx, sk, w);
            const uint32_t mk = __ballot_sync(0xFFFFFFFFu, go);
            if (go) q2[n2 + __popc(mk & lt)] = w;
            n2 += __popc(mk);
            if (has_old) n2_old = n2;  // conservatively: everything queued so far may be old
            __syncwarp();
            if (n2 >= 32u) run_level2(32u);
        };
        // full batches from the front of Q1; the leftover (< 32) moves to the front
        auto run_batches = [&]() {
            uint32_t head = 0;
            while (n1 - head >= 32u) {
                run_level1(head, 32u, head < n1_old);
                head += 32u;
            }
            if (head) {
                const uint32_t left = n1 - head;
                uint32_t e = 0;
                if ((uint32_t)lane < left) e = q1[head + lane];
                __syncwarp();
                if ((uint32_t)lane < left) q1[lane] = e;
                __syncwarp();
                n1 = left;
                n1_old = 0;
            }
        };

        if (n_steps) mbar_wait(bar_full, 0u);
        for (uint32_t s = 0; s < n_steps; ++s) {
            mbar_wait(bar_full + 8u * slot, use & 1u);
            if (group < g.n_groups) {
                const int pos = (int)slot * RC + 4 * rho;  // ring row of this warp's active row
                const uint8_t* rowp = ring0 + pos * pitch + kBandHaloB + colb;
                uint4 wc = make_uint4(0, 0, 0, 0), wu = wc, wd = wc;
                uint32_t pv = 0, nx = 0;
                if (in) {
                    wc = *reinterpret_cast<const uint4*>(rowp);
                    wu = *reinterpret_cast<const uint4*>(rowp - pitch + (pos == 0 ? cx.ring_bytes : 0));
                    wd = *reinterpret_cast<const uint4*>(rowp + pitch);
                    pv = *reinterpret_cast<const uint32_t*>(rowp - 4);
                    nx = *reinterpret_cast<const uint32_t*>(rowp + 16);
                }
                const uint32_t c4[4] = {wc.x, wc.y, wc.z, wc.w};
                const uint32_t u4[4] = {wu.x, wu.y, wu.z, wu.w};
                const uint32_t d4[4] = {wd.x, wd.y, wd.z, wd.w};
                const uint32_t ebase = (par << 31) | ((uint32_t)pos << 16);
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
#pragma unroll
                        for (int w = 0; w < 4; ++w) {
                            const bool pred = nb[w] != 0u;
                            const uint32_t mk = __ballot_sync(0xFFFFFFFFu, pred);
                            if (pred) q1[n1 + __popc(mk & lt)] = ebase | (uint32_t)(colb + 4 * w + cj);
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
#pragma unroll
                            for (int bb = 0; bb < 8; ++bb) {
                                const int bit = cj + 4 * bb;
                                const bool pred = (nb[w] >> bit) & 1u;
                                const uint32_t mk = __ballot_sync(0xFFFFFFFFu, pred);
                                if (pred) q1[n1 + __popc(mk & lt)] = ebase | (uint32_t)(8 * (colb + 4 * w) + bit);
                                n1 += __popc(mk);
                            }
                            __syncwarp();
                            run_batches();
                        }
                    }
                }
            }
            // sites queued by step s-1 must be finished now: their rows are about to be released
            if (n1_old) {  // then n1 < 32
                run_level1(0u, n1, true);
                n1 = 0;
            }
            if (n2_old) run_level2(n2);  // then n2 < 32
            if (s > 0) {
                if (lane == 0) mbar_arrive(bar_empty + 8u * rel_slot);  // chunk s-1 is free
                if (++rel_slot == NS) rel_slot = 0;
            }
            n1_old = n1;
            n2_old = n2;
            par ^= 1u;
            grow_cur += RC;
            group += g.R;
            if (++slot == NS) { slot = 0; ++use; }
        }
        // drain: everything left was queued by the last step
        par ^= 1u;
        grow_cur -= RC;
        if (n1) {
            run_level1(0u, n1, true);
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
inline bool band_supported(int fmt, uint32_t L)
{
    if (L >= 65536) return false;
    return fmt == kFmtU8 ? (L % 16 == 0) : (L % 128 == 0);  // rows are multiples of 16 bytes
}

inline int band_plan(int fmt, uint32_t L, uint32_t B, BandPlan* p)
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
        e = cudaFuncSetAttribute(phase_band_kernel<kFmtU8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 1024);
        if (e != cudaSuccess) return (int)e;
        e = cudaFuncSetAttribute(phase_band_kernel<kFmtBits>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 1024);
        if (e != cudaSuccess) return (int)e;
        sm_count = sms;
    }
    p->row_bytes = fmt == kFmtU8 ? L : L / 8;
    const uint32_t tasks = (p->row_bytes + kBandTaskB - 1) / kBandTaskB;
    uint32_t tpr_log2 = 0;
    while ((1u << tpr_log2) < tasks && tpr_log2 < 4) ++tpr_log2;
    p->tpr_log2 = tpr_log2;
    p->W = (1u << tpr_log2) * kBandTaskB;
    p->n_strips = (p->row_bytes + p->W - 1) / p->W;
    p->R = kBandConsumers >> tpr_log2;
    p->RC = 4 * p->R;
    p->pitch = p->W + 2 * kBandHaloB;
    p->slot_bytes = p->RC * p->pitch;
    p->n_groups = L / 4;
    p->n_super = (p->n_groups + p->R - 1) / p->R;
    uint32_t per_strip = (uint32_t)sm_count / (p->n_strips * B);
    if (per_strip < 1) per_strip = 1;
    p->nb = p->n_super < per_strip ? p->n_super : per_strip;
    const uint32_t max_chunks = (p->n_super + p->nb - 1) / p->nb + 1;
    uint32_t want = kBandMaxSlots;
    if (const char* e = getenv("PGG_BAND_SLOTS")) want = (uint32_t)atoi(e);
    if (want > (uint32_t)kBandMaxSlots) want = kBandMaxSlots;
    if (want < 3) want = 3;
    const uint32_t fixed = fmt == kFmtU8 ? band_fixed_bytes<kFmtU8>() : band_fixed_bytes<kFmtBits>();
    while (want > 3 && want * p->slot_bytes + fixed > (uint32_t)smem_optin - 1024) --want;
    if (max_chunks < want) want = max_chunks < 3 ? 3 : max_chunks;
    p->NS = want;
    p->smem_bytes = p->NS * p->slot_bytes + fixed;
    return 0;
}

inline void band_launch(const BandPlan& p, int fmt, const PhaseArgs& a, uint32_t m, uint32_t k,
                        uint32_t B, cudaStream_t stream)
{
    static const bool pdl = [] { const char* e = getenv("PGG_PDL"); return e == nullptr || atoi(e) != 0; }();
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(p.n_strips * p.nb, B);
    cfg.blockDim = dim3(kBandThreads);
    cfg.dynamicSmemBytes = p.smem_bytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (fmt == kFmtU8)
        cudaLaunchKernelEx(&cfg, phase_band_kernel<kFmtU8>, a, m, k, p);
    else
        cudaLaunchKernelEx(&cfg, phase_band_kernel<kFmtBits>, a, m, k, p);
}

}  // namespace pgg
