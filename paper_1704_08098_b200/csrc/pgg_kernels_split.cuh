// pgg_kernels_split.cuh -- the SPLIT phase kernel (K1, uint8): the RING kernel's data
// movement and arithmetic with the consumer work divided between two kinds of warps.
//
// ncu on RING at L = 16384 (profiles/r1_ring_u8_late.md): with six ring slots the stream
// alone would finish a phase in 43 us, but the 16 consumer warps (4 per scheduler; the
// 227 KB ring leaves room for one CTA per SM) issue only 0.58 instructions per cycle
// and scheduler: every warp walks the same dependent chain scan -> compaction -> Philox
// -> stencil.  SPLIT puts 25 warps on the SM (80 registers each):
//
//   warp 24      producer: bulk-async copies of row chunks into the ring (as in RING)
//   warps 16-23  scanners: scanner i scans column tasks 2i and 2i+1 of every step (S9
//                bulk test, ballot compaction) and appends the surviving sites to the
//                queues of workers 2i and 2i+1
//   warps 0-15   workers: worker w pops batches of 32 (or 64) sites from its queue and
//                runs Philox, the neighbour compare, the 14-read stencil A_x - A_y, the
//                threshold compare and the in-place write (ring_level1 / ring_level2)
//
// A queue is a single-producer single-consumer ring of kSplitQCap (soff, site) entries in
// shared memory.  The scanner publishes, once per step, the running entry count of each of
// its two queues (tails[w][s & 7]) and then the step number (posted[i] = s + 1, st.release);
// the worker polls posted (ld.acquire), publishes its running consumed count (heads[w]) for
// the scanner's space check, and -- as in RING -- releases chunk s-1 once every site queued
// in steps <= s-1 is finished, so a leftover (< 32) waits for the next step's sites.
// All counters are monotonic: no phase-parity aliasing between the two sides.
#pragma once
#include "pgg_kernels_ring.cuh"

namespace pgg {

constexpr int kSplitWorkers = 16;
constexpr int kSplitScanners = 8;
constexpr int kSplitThreads = (kSplitWorkers + kSplitScanners + 1) * 32;
constexpr int kSplitQCap = 160;  // entries per queue: leftover (< 32) + the 128 sites of one task
constexpr int kSplitCtlWords = kSplitWorkers * 8 + kSplitWorkers + kSplitScanners;  // tails, heads, posted
constexpr int kSplitFixedBytes = kSplitWorkers * kSplitQCap * 8 + kSplitCtlWords * 4 + 160 * 4
                               + 2 * kRingMaxSlots * 8 + 8 * 4 + 128;

__device__ __forceinline__ uint32_t lds_acquire(const uint32_t* p)
{
    uint32_t v;
    asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ void sts_release(uint32_t* p, uint32_t v)
{
    asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}

__global__ void __launch_bounds__(kSplitThreads, 1)
phase_split_kernel(PhaseArgs a, uint32_t m, uint32_t k, RingPlan g)
{
    constexpr int FMT = kFmtU8;
    extern __shared__ __align__(128) uint8_t smem_raw[];
    const uint32_t NS = g.NS;
    const int RC = (int)g.RC, pitch = (int)g.pitch;
    uint8_t* ring0 = smem_raw;
    uint2* queues = reinterpret_cast<uint2*>(ring0 + (size_t)NS * g.slot_bytes);
    uint32_t* tails = reinterpret_cast<uint32_t*>(queues + kSplitWorkers * kSplitQCap);  // [16][8]
    uint32_t* heads = tails + kSplitWorkers * 8;                                          // [16]
    uint32_t* posted = heads + kSplitWorkers;                                             // [8]
    uint32_t* tbl = posted + kSplitScanners;
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(tbl + 160);  // full[NS], empty[NS]
    int* eoff = reinterpret_cast<int*>(bars + 2 * kRingMaxSlots);                 // e[4], f[4]
    __shared__ int delta_cta;

    const uint32_t b = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t L = a.L;
    const uint32_t cls = a.order[((size_t)b * a.order_stride + (m % a.order_stride)) * 16 + k];
    const int ci = (int)(cls >> 2), cj = (int)(cls & 3u);
    uint8_t* lat = a.lats + (size_t)b * a.lat_bytes;
    const uint32_t bar_full = smem_u32(bars), bar_empty = bar_full + 8u * NS;

    for (int q = threadIdx.x; q < kTableSize; q += kSplitThreads)
        tbl[q] = a.tables[(size_t)b * kTableSize + q];
    for (int q = threadIdx.x; q < kSplitCtlWords; q += kSplitThreads) tails[q] = 0u;
    if (threadIdx.x == 0) {
        delta_cta = 0;
        for (uint32_t s = 0; s < NS; ++s) {
            mbar_init(bar_full + 8u * s, 1);
            mbar_init(bar_empty + 8u * s, kSplitWorkers);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        eoff[0] = -pitch; eoff[1] = pitch; eoff[2] = -1;    eoff[3] = 1;
        eoff[4] = 1;      eoff[5] = 1;     eoff[6] = pitch; eoff[7] = pitch;
    }
    __syncthreads();

    const uint32_t strip = blockIdx.x / g.nb, band = blockIdx.x - strip * g.nb;
    const uint32_t S0 = (uint32_t)(((unsigned long long)band * g.n_super) / g.nb);
    const uint32_t S1 = (uint32_t)(((unsigned long long)(band + 1) * g.n_super) / g.nb);
    const uint32_t n_steps = S1 - S0;
    const int j0b = (int)(strip * g.W);
    const int wb = min((int)g.W, (int)g.row_bytes - j0b);  // core bytes per row of this strip
    const int slot_bytes = (int)g.slot_bytes;
    const int ring_bytes = (int)NS * slot_bytes;

    if (warp == kSplitWorkers + kSplitScanners) {
        // ---------------- producer warp (as in RING, no mirror rows) ----------------
        const int rb = (int)g.row_bytes;
        const bool left_edge = j0b == 0, right_edge = j0b + wb == rb;
        const uint32_t ring_s = smem_u32(ring0);
        const uint32_t n_chunks = n_steps ? n_steps + 1 : 0;
        const uint32_t row_tx = (uint32_t)(wb + 2 * kRingHaloB);
        // first lattice row of chunk kc: the first active row of step S0 + kc - 1 (mod L)
        int row0 = (int)(((long long)RC * ((long long)S0 - 1) + ci) % (long long)L);
        if (row0 < 0) row0 += (int)L;
        uint32_t slot = 0, use = 0;  // chunk kc lives in slot kc % NS, use = kc / NS
        for (uint32_t kc = 0; kc < n_chunks; ++kc) {
            if (use > 0) mbar_wait(bar_empty + 8u * slot, (use - 1u) & 1u);
            const uint32_t bar = bar_full + 8u * slot;
            const int r_lo = kc == 0 ? RC - 3 : 0;  // of the prologue chunk only the tail is read
            if (lane == 0) mbar_expect_tx(bar, (uint32_t)(RC - r_lo) * row_tx);
            __syncwarp();
            for (int rr = r_lo + lane; rr < RC; rr += 32) {
                const int gi = (int)((uint32_t)(row0 + rr) % L);
                const uint8_t* src = lat + (size_t)gi * (size_t)rb;
                const uint32_t dst = ring_s + (slot * (uint32_t)RC + (uint32_t)rr) * (uint32_t)pitch;
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
    } else if (warp >= kSplitWorkers) {
        // ---------------- scanner warps ----------------
        const int sc = warp - kSplitWorkers;
        const uint32_t lt = (1u << lane) - 1u;
        const int tmask = (1 << g.tpr_log2) - 1;
        uint32_t slot = 1 % NS, par = (1 / NS) & 1u;  // of chunk s + 1, and its "full" parity
        // per column task h (worker 2 sc + h): this lane's 16 bytes of the task's active row
        // (byte offset from ring0), the lattice site index of the first of them, the running
        // entry count of the worker's queue and its write index
        int rowoff[2], up_wrapped[2], upoff[2];
        uint32_t site0[2], n_act[2], tail[2] = {0u, 0u}, tidx[2] = {0u, 0u};
        bool in[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int t = 2 * sc + h, rho = t >> g.tpr_log2, tau = t & tmask;
            const int colb = tau * kRingTaskB + 16 * lane;
            in[h] = colb < wb;
            rowoff[h] = (int)slot * slot_bytes + 4 * rho * pitch + kRingHaloB + colb;
            up_wrapped[h] = rho != 0 ? -pitch : ring_bytes - pitch;
            upoff[h] = slot == 0 ? up_wrapped[h] : -pitch;
            site0[h] = (uint32_t)(RC * (int)S0 + 4 * rho + ci) * L + (uint32_t)(j0b + colb);
            const uint32_t first_group = S0 * g.R + (uint32_t)rho;
            n_act[h] = first_group >= g.n_groups ? 0u
                     : min(n_steps, (g.n_groups - first_group + g.R - 1) / g.R);
        }
        const uint32_t site_step = (uint32_t)RC * L;
        const uint32_t bm = 0xFFu << (8 * cj);

        if (n_steps) mbar_wait(bar_full, 0u);  // the prologue chunk (the rows above the first active row)
        for (uint32_t s = 0; s < n_steps; ++s) {
            mbar_wait(bar_full + 8u * slot, par);
            uint32_t nb[2][4];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                uint4 wc = make_uint4(0, 0, 0, 0), wu = wc, wd = wc;
                uint32_t pv = 0, nx = 0;
                if (in[h] && s < n_act[h]) {
                    const uint8_t* rowp = ring0 + rowoff[h];
                    wc = *reinterpret_cast<const uint4*>(rowp);
                    wu = *reinterpret_cast<const uint4*>(rowp + upoff[h]);
                    wd = *reinterpret_cast<const uint4*>(rowp + pitch);
                    pv = *reinterpret_cast<const uint32_t*>(rowp - 4);
                    nx = *reinterpret_cast<const uint32_t*>(rowp + 16);
                }
                const uint32_t c4[4] = {wc.x, wc.y, wc.z, wc.w};
                const uint32_t u4[4] = {wu.x, wu.y, wu.z, wu.w};
                const uint32_t d4[4] = {wd.x, wd.y, wd.z, wd.w};
#pragma unroll
                for (int w = 0; w < 4; ++w) {
                    // word w = sites 4w..4w+3 of this lane's 16; the active one is byte cj
                    const uint32_t lw = __funnelshift_l(w == 0 ? pv : c4[w - 1], c4[w], 8);
                    const uint32_t rw = __funnelshift_r(c4[w], w == 3 ? nx : c4[w + 1], 8);
                    nb[h][w] = ((c4[w] ^ u4[w]) | (c4[w] ^ d4[w]) | (c4[w] ^ lw) | (c4[w] ^ rw)) & bm;  // S9
                }
            }
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (__any_sync(0xFFFFFFFFu, (nb[h][0] | nb[h][1] | nb[h][2] | nb[h][3]) != 0u)) {
                    uint32_t mk[4], cnt = 0;
#pragma unroll
                    for (int w = 0; w < 4; ++w) {
                        mk[w] = __ballot_sync(0xFFFFFFFFu, nb[h][w] != 0u);
                        cnt += __popc(mk[w]);
                    }
                    // space: the worker has consumed heads[] entries; at most kSplitQCap may be pending
                    const uint32_t* hp = heads + 2 * sc + h;
                    while (tail[h] + cnt - lds_acquire(hp) > (uint32_t)kSplitQCap) __nanosleep(40);
                    uint2* q = queues + (2 * sc + h) * kSplitQCap;
                    const uint32_t so = (uint32_t)(rowoff[h] + cj), si = site0[h] + (uint32_t)cj;
                    uint32_t at = tidx[h];
#pragma unroll
                    for (int w = 0; w < 4; ++w) {
                        if (nb[h][w] != 0u) {
                            uint32_t idx = at + __popc(mk[w] & lt);
                            idx = idx >= (uint32_t)kSplitQCap ? idx - kSplitQCap : idx;
                            q[idx] = make_uint2(so + 4u * w, si + 4u * w);
                        }
                        at += __popc(mk[w]);
                    }
                    tail[h] += cnt;
                    tidx[h] = at >= (uint32_t)kSplitQCap ? at - kSplitQCap : at;
                }
            }
            __syncwarp();
            if (lane == 0) {
                tails[(2 * sc) * 8 + (s & 7u)] = tail[0];
                tails[(2 * sc + 1) * 8 + (s & 7u)] = tail[1];
                sts_release(posted + sc, s + 1u);
            }
            const bool wrapnow = slot + 1 == NS;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                site0[h] += site_step;
                rowoff[h] += wrapnow ? slot_bytes - ring_bytes : slot_bytes;
                upoff[h] = wrapnow ? up_wrapped[h] : -pitch;
            }
            if (wrapnow) { slot = 0; par ^= 1u; } else ++slot;
        }
    } else {
        // ---------------- worker warps ----------------
        const int w = warp, sc = w >> 1;
        const StepKey sk = make_step_key(a.seeds[b], a.t_begin + m, k, cls);
        const uint2* q = queues + w * kSplitQCap;
        const int wrap = ring_bytes, wrap_below = pitch;  // sites of ring row 0 take the wrapping stencil
        uint32_t head = 0, hidx = 0, prevT = 0, T = 0, rel_slot = 0;
        uint32_t slot = 1 % NS, par = (1 / NS) & 1u;  // of chunk s + 1, and its "full" parity
        int delta = 0;
        // one site per lane: draw + neighbour compare, stencil + accept + write for the lanes that go on
        auto one = [&](uint32_t idx) {
            idx = idx >= (uint32_t)kSplitQCap ? idx - kSplitQCap : idx;
            uint4 v;
            if (ring_level1<FMT>(q[idx], ring0, eoff, sk, v, wrap))
                delta += ring_level2<FMT>(v, ring0, eoff, lat, tbl, wrap, wrap_below);
        };
        auto advance = [&](uint32_t cnt) {
            head += cnt;
            hidx += cnt;
            hidx = hidx >= (uint32_t)kSplitQCap ? hidx - kSplitQCap : hidx;
        };
        if (n_steps) mbar_wait(bar_full, 0u);
        for (uint32_t s = 0; s < n_steps; ++s) {
            while (lds_acquire(posted + sc) <= s) __nanosleep(40);
            // the scanner has seen this chunk arrive; observing its barrier here as well makes the
            // bulk-async writes visible to this warp's own reads (no wait: the phase is complete)
            mbar_wait(bar_full + 8u * slot, par);
            if (++slot == NS) { slot = 0; par ^= 1u; }
            T = tails[w * 8 + (s & 7u)];
            while (T - head >= 64u) {  // two independent Philox chains per lane
                uint4 va, vb;
                uint32_t ia = hidx + lane, ib = hidx + 32 + lane;
                ia = ia >= (uint32_t)kSplitQCap ? ia - kSplitQCap : ia;
                ib = ib >= (uint32_t)kSplitQCap ? ib - kSplitQCap : ib;
                const bool ga = ring_level1<FMT>(q[ia], ring0, eoff, sk, va, wrap);
                const bool gb = ring_level1<FMT>(q[ib], ring0, eoff, sk, vb, wrap);
                if (ga) delta += ring_level2<FMT>(va, ring0, eoff, lat, tbl, wrap, wrap_below);
                if (gb) delta += ring_level2<FMT>(vb, ring0, eoff, lat, tbl, wrap, wrap_below);
                advance(64u);
            }
            if (T - head >= 32u) {
                one(hidx + lane);
                advance(32u);
            }
            if (head < prevT) {  // sites queued by step s-1 are still waiting: their rows go now
                const uint32_t cnt = T - head;  // < 32
                if ((uint32_t)lane < cnt) one(hidx + lane);
                advance(cnt);
            }
            __syncwarp();  // every lane has read its entries
            if (lane == 0) {
                sts_release(heads + w, head);
                if (s > 0) mbar_arrive(bar_empty + 8u * rel_slot);  // chunk s-1 is free
            }
            if (s > 0 && ++rel_slot == NS) rel_slot = 0;
            prevT = T;
        }
        // drain: everything left was queued by the last step
        if ((uint32_t)lane < T - head) one(hidx + lane);
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
// Host side: RING's geometry (ring_plan) with SPLIT's fixed shared-memory part
// ---------------------------------------------------------------------------
inline bool split_supported(int fmt, uint32_t L)
{
    return fmt == kFmtU8 && ring_supported(fmt, L);
}

inline int split_plan(uint32_t L, uint32_t B, RingPlan* p)
{
    int smem_optin = 0;  // per call (the function attribute is per device)
    {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaFuncSetAttribute(phase_split_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 256);
        if (e != cudaSuccess) return (int)e;
    }
    int rc = ring_plan(kFmtU8, L, B, p, false);
    if (rc != 0) return rc;
    p->mirror = 0;
    const uint32_t max_chunks = (p->n_super + p->nb - 1) / p->nb + 1;
    uint32_t want = kRingMaxSlots;
    if (const char* e = getenv("PGG_RING_SLOTS")) want = (uint32_t)atoi(e);
    if (want > (uint32_t)kRingMaxSlots) want = kRingMaxSlots;
    if (want < 3) want = 3;
    while (want > 3 && want * p->slot_bytes + kSplitFixedBytes > (uint32_t)smem_optin - 256) --want;
    if (max_chunks < want) want = max_chunks < 3 ? 3 : max_chunks;
    p->NS = want;
    p->smem_bytes = p->NS * p->slot_bytes + kSplitFixedBytes;
    return 0;
}

inline void split_launch(const RingPlan& p, const PhaseArgs& a, uint32_t m, uint32_t k, uint32_t B,
                         cudaStream_t stream)
{
    dim3 grid(p.n_strips * p.nb, B);
    phase_split_kernel<<<grid, kSplitThreads, p.smem_bytes, stream>>>(a, m, k, p);
}

}  // namespace pgg
