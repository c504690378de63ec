// pgg_kernels_band.cuh -- the BAND phase kernel (K1 uint8, K2 bit-packed).
//
// Measured on B200 (profiles/): cp.async.bulk copies of ~0.5 KB issued by one
// warp deliver only ~2.2 TB/s chip-wide, copies of >= 1 KB reach 5.6-5.8 TB/s.
// So the lattice is not cut into square tiles (short rows, 16 % halo re-reads)
// but into column STRIPS of up to 8 KB, and every persistent CTA streams one
// BAND of consecutive lattice rows of a strip through a ring of row chunks in
// shared memory: each lattice row is fetched exactly once per phase by one
// large bulk-async copy (SASS UBLKCP, completing on an mbarrier), plus 16
// bytes of column halo on each side (3 sites are needed; 16 bytes keep every
// copy 16-byte aligned; at the lattice edge the halo is the periodic image).
//
//   ring   = [mirror: 3 rows][slot 0][slot 1]...[slot NS-1], slot = RC rows
//   chunk k of a band = RC = 4 R consecutive lattice rows, first row = an
//            active row (row % 4 == ci); lives in slot k % NS.
//   step s  = the R active rows of chunk s+1; their stencils reach 3 rows up
//            (tail of chunk s) and 3 rows down (inside chunk s+1).
//   mirror = copy of the last 3 rows of slot NS-1 placed in front of slot 0,
//            written by the producer warp, so that the 7-row window of every
//            active row is contiguous in shared memory.
//
// 16 consumer warps: warp w owns 128 active sites (uint8; 512 bytes) or 1024
// (bit-packed) of active row w / tpr, column task w % tpr, of every step.
// Scan (S9 bulk test, word-wide logic), per-warp compaction queue, batches of
// 32 through Philox + stencil + accept as in pgg_kernels_pipe.cuh.  A warp
// releases chunk s-1 at the end of step s, so leftovers (< 32 queued sites) of
// step s-1 are batched with the sites of step s.
#pragma once
#include "pgg_kernels_pipe.cuh"

namespace pgg {

constexpr int kBandConsumers = 16;
constexpr int kBandThreads = (kBandConsumers + 1) * 32;
constexpr int kBandTaskB = 512;     // bytes of one lattice row that one warp scans per step
constexpr int kBandHaloB = 16;
constexpr int kBandQueueCap = 512;  // ring entries per warp (power of two)
constexpr int kBandMaxSlots = 6;
constexpr int kBandFixedBytes = kBandConsumers * kBandQueueCap * 4 + 160 * 4 + (2 * kBandMaxSlots + 2) * 8 + 128;

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

// Steps a3-a7 for one queued site; entry = step parity << 31 | ring row << 16 | site column.
template <int FMT>
__device__ __forceinline__ int band_process(uint32_t e, uint32_t par_cur, const uint8_t* __restrict__ ring0,
                                            int pitch, int rc_mask, int grow_cur, int grow_prev, int j0,
                                            uint8_t* __restrict__ lat, uint32_t L, const StepKey& sk,
                                            const uint32_t* __restrict__ tbl)
{
    const int pos = (int)((e >> 16) & 0x7FFFu), c = (int)(e & 0xFFFFu);
    const int gi = (((e >> 31) == par_cur) ? grow_cur : grow_prev) + (pos & rc_mask);
    const uint32_t site = (uint32_t)gi * L + (uint32_t)(j0 + c);
    uint32_t x0, u;
    step_draw(sk, site, x0, u);
    const uint32_t dir = x0 >> 30;  // 0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1)
    // e = unit step towards y, f = perpendicular unit step (ring row, site column)
    const int er = dir == 0 ? -1 : dir == 1 ? 1 : 0;
    const int ec = dir == 2 ? -1 : dir == 3 ? 1 : 0;
    const int fr = dir < 2 ? 0 : 1, fc = dir < 2 ? 1 : 0;
    int sx, sy, dA;
    if (FMT == kFmtU8) {
        const uint8_t* p = ring0 + pos * pitch + kBandHaloB + c;
        const int eo = er * pitch + ec, fo = fr * pitch + fc;
        sx = p[0];
        sy = p[eo];
        if (sx == sy) return 0;
        // A_x - A_y with A = 5 s + 2 (nearest + diagonal) + axial distance-2 (include/pgg.h):
        // weights of x's 13-site stencil minus those of y's, at offset (a along e, b along f)
        dA = p[-2 * eo] + p[-eo] - p[2 * eo] - p[3 * eo] + 3 * (sx - sy)
           + 2 * (p[-eo + fo] + p[-eo - fo] - p[2 * eo + fo] - p[2 * eo - fo])
           + p[2 * fo] + p[-2 * fo] - p[eo + 2 * fo] - p[eo - 2 * fo];
    } else {
        const uint8_t* rowp = ring0 + pos * pitch;
        const int cc = c + 8 * kBandHaloB;
        auto S = [&](int a, int b) {
            const int rr = a * er + b * fr, q = cc + a * ec + b * fc;
            return (int)((rowp[rr * pitch + (q >> 3)] >> (q & 7)) & 1);
        };
        sx = S(0, 0);
        sy = S(1, 0);
        if (sx == sy) return 0;
        dA = S(-2, 0) + S(-1, 0) - S(2, 0) - S(3, 0) + 3 * (sx - sy)
           + 2 * (S(-1, 1) + S(-1, -1) - S(2, 1) - S(2, -1))
           + S(0, 2) + S(0, -2) - S(1, 2) - S(1, -2);
    }
    if (u < tbl[table_index(dA, sx - sy)]) {
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
    const uint32_t NS = g.NS;
    uint8_t* ring0 = smem_raw + 3 * g.pitch;  // slot 0, row 0; the mirror sits in front of it
    uint32_t* queues = reinterpret_cast<uint32_t*>(smem_raw + 3 * g.pitch + (size_t)NS * g.slot_bytes);
    uint32_t* tbl = queues + kBandConsumers * kBandQueueCap;
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(tbl + 160);  // full[NS], empty[NS], mirror
    __shared__ int delta_cta;

    const uint32_t b = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t L = a.L;
    const uint32_t cls = a.order[((size_t)b * a.order_stride + (m % a.order_stride)) * 16 + k];
    const int ci = (int)(cls >> 2), cj = (int)(cls & 3u);
    uint8_t* lat = a.lats + (size_t)b * a.lat_bytes;
    const uint32_t bar_full = smem_u32(bars), bar_empty = bar_full + 8u * NS, bar_mirror = bar_full + 16u * NS;

    for (int q = threadIdx.x; q < kTableSize; q += kBandThreads)
        tbl[q] = a.tables[(size_t)b * kTableSize + q];
    if (threadIdx.x == 0) {
        delta_cta = 0;
        for (uint32_t s = 0; s < NS; ++s) {
            mbar_init(bar_full + 8u * s, 1);
            mbar_init(bar_empty + 8u * s, kBandConsumers);
        }
        mbar_init(bar_mirror, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

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
            // chunk kc just went to slot 0: mirror the tail of slot NS-1 (chunk kc-1) in front of it
            // (the mirror's previous readers released chunk kc-1-NS, which this warp waited for
            // before it re-armed slot NS-1)
            if (kc >= 1 && slot == 0) {
                mbar_wait(bar_full + 8u * (NS - 1u), (use - 1u) & 1u);
                const uint4* srcm = reinterpret_cast<const uint4*>(ring0 + (size_t)NS * g.slot_bytes - 3 * pitch);
                uint4* dstm = reinterpret_cast<uint4*>(smem_raw);
                const int n16 = 3 * pitch / 16;
                int i = lane;
                for (; i + 7 * 32 < n16; i += 8 * 32) {
                    uint4 v[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j) v[j] = srcm[i + 32 * j];
#pragma unroll
                    for (int j = 0; j < 8; ++j) dstm[i + 32 * j] = v[j];
                }
                for (; i < n16; i += 32) dstm[i] = srcm[i];
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_mirror);
            }
            row0 += RC;
            if (row0 >= (int)L) row0 %= (int)L;
            if (++slot == NS) { slot = 0; ++use; }
        }
    } else {
        // ---------------- consumer warps ----------------
        const StepKey sk = make_step_key(a.seeds[b], a.t_begin + m, k, cls);
        uint32_t* q = queues + warp * kBandQueueCap;
        const uint32_t lt = (1u << lane) - 1u;
        const int rho = warp >> g.tpr_log2, tau = warp & ((1 << g.tpr_log2) - 1);
        const int colb = tau * kBandTaskB + 16 * lane;  // first core byte of this lane's 16
        const bool in = colb < wb;
        const int j0 = (FMT == kFmtU8) ? j0b : j0b * 8;
        const int rc_mask = RC - 1;
        // the queue is linear: entries [0, qn); the first n_prev of them were queued by the previous step
        uint32_t qn = 0, n_prev = 0;
        int delta = 0;
        uint32_t slot = 1 % NS, use = 1 / NS;       // of chunk s + 1
        uint32_t rel_slot = 0;                      // slot of chunk s - 1
        uint32_t mir_par = 0;
        int grow_cur = RC * (int)S0 + ci;           // lattice row of the step's first active row
        uint32_t group = S0 * g.R + (uint32_t)rho;  // index of this warp's active row among the class rows

        auto run_batches = [&](uint32_t par) {
            // full batches from the front; the leftover (< 32) moves to the front
            uint32_t head = 0;
            while (qn - head >= 32u) {
                delta += band_process<FMT>(q[head + lane], par, ring0, pitch, rc_mask, grow_cur, grow_cur - RC, j0,
                                           lat, L, sk, tbl);
                head += 32u;
            }
            if (head) {
                const uint32_t left = qn - head;
                uint32_t e = 0;
                if ((uint32_t)lane < left) e = q[head + lane];
                __syncwarp();
                if ((uint32_t)lane < left) q[lane] = e;
                __syncwarp();
                qn = left;
                n_prev = 0;
            }
        };

        if (n_steps) mbar_wait(bar_full, 0u);
        for (uint32_t s = 0; s < n_steps; ++s) {
            const uint32_t par = s & 1u;
            mbar_wait(bar_full + 8u * slot, use & 1u);
            if (slot == 0) {
                mbar_wait(bar_mirror, mir_par);
                mir_par ^= 1u;
            }
            if (group < g.n_groups) {
                const int pos = (int)slot * RC + 4 * rho;  // ring row of this warp's active row
                const uint8_t* rowp = ring0 + pos * pitch + kBandHaloB + colb;
                uint4 wc = make_uint4(0, 0, 0, 0), wu = wc, wd = wc;
                uint32_t pv = 0, nx = 0;
                if (in) {
                    wc = *reinterpret_cast<const uint4*>(rowp);
                    wu = *reinterpret_cast<const uint4*>(rowp - pitch);
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
                            if (pred) q[qn + __popc(mk & lt)] = ebase | (uint32_t)(colb + 4 * w + cj);
                            qn += __popc(mk);
                        }
                        __syncwarp();
                        run_batches(par);
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
                                if (pred) q[qn + __popc(mk & lt)] = ebase | (uint32_t)(8 * (colb + 4 * w) + bit);
                                qn += __popc(mk);
                            }
                            __syncwarp();
                            run_batches(par);
                        }
                    }
                }
            }
            // sites of step s-1 still queued (then fewer than 32 are queued in all): flush them
            if (n_prev) {
                if ((uint32_t)lane < qn)
                    delta += band_process<FMT>(q[lane], par, ring0, pitch, rc_mask, grow_cur, grow_cur - RC, j0, lat, L,
                                               sk, tbl);
                qn = 0;
            }
            __syncwarp();
            if (s > 0) {
                if (lane == 0) mbar_arrive(bar_empty + 8u * rel_slot);  // chunk s-1 is free
                if (++rel_slot == NS) rel_slot = 0;
            }
            n_prev = qn;
            grow_cur += RC;
            group += g.R;
            if (++slot == NS) { slot = 0; ++use; }
        }
        // drain: everything left was queued by the last step
        if (qn) {
            if ((uint32_t)lane < qn)
                delta += band_process<FMT>(q[lane], (n_steps - 1u) & 1u, ring0, pitch, rc_mask, grow_cur - RC,
                                           grow_cur - 2 * RC, j0, lat, L, sk, tbl);
        }
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
    static int sm_count = 0, smem_optin = 0;
    if (sm_count == 0) {
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
    uint32_t want = 5;
    if (const char* e = getenv("PGG_BAND_SLOTS")) want = (uint32_t)atoi(e);
    if (want > (uint32_t)kBandMaxSlots) want = kBandMaxSlots;
    if (want < 3) want = 3;
    while (want > 3 && 3 * p->pitch + want * p->slot_bytes + kBandFixedBytes > (uint32_t)smem_optin - 1024) --want;
    if (max_chunks < want) want = max_chunks < 3 ? 3 : max_chunks;
    p->NS = want;
    p->smem_bytes = 3 * p->pitch + p->NS * p->slot_bytes + kBandFixedBytes;
    return 0;
}

inline void band_launch(const BandPlan& p, int fmt, const PhaseArgs& a, uint32_t m, uint32_t k,
                        uint32_t B, cudaStream_t stream)
{
    dim3 grid(p.n_strips * p.nb, B);
    if (fmt == kFmtU8)
        phase_band_kernel<kFmtU8><<<grid, kBandThreads, p.smem_bytes, stream>>>(a, m, k, p);
    else
        phase_band_kernel<kFmtBits><<<grid, kBandThreads, p.smem_bytes, stream>>>(a, m, k, p);
}

}  // namespace pgg
