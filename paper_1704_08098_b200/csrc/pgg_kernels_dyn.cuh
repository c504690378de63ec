// pgg_kernels_dyn.cuh -- the DYN phase kernel (K1, uint8): the RING kernel with its work
// handed out dynamically, so that more than 16 consumer warps fit one step.
//
// RING ties consumer warp w to column task w of every step (16 tasks of 512 bytes per
// step), which fixes the SM at 17 warps -- 4 per scheduler, 0.58 instructions per cycle
// (profiles/r1_ring_u8_late.md) -- and makes every step as slow as its busiest column.
// Here the (step, task) pairs of a band are numbered g = 16 s + task and NW consumer
// warps (24 by default) draw the next g from a shared-memory counter.  A warp handles its
// task exactly as a RING warp handles one step of its column: scan (S9), ballot
// compaction into its own queue, Philox batches of 32 / 64, inline stencil, in-place
// write.  A leftover of fewer than 32 queued sites rides along with the warp's NEXT task
// (whatever step that is), as in RING.
//
// Ring-slot release is counted per task instead of per warp: chunk c is read by the 16
// tasks of step c-1 (their active rows) and by the 16 tasks of step c (the three rows
// above theirs), so its "empty" mbarrier expects 32 arrivals, two from every finished
// task (chunk 0, the prologue rows, gets 16 of them at initialisation).  A task is
// finished when none of its sites is queued any more.  A warp never waits for a chunk
// whose load can depend on its own unfinished task: before taking a task NS-2 or more
// steps ahead of the one it still holds sites of, it runs those as a partial batch.
#pragma once
#include "pgg_kernels_ring.cuh"

namespace pgg {

constexpr int kDynQ1Cap = 160;  // 8-byte entries per warp: leftover (< 32) + 128 new

template <int NW>
constexpr int dyn_fixed_bytes()
{
    return NW * kDynQ1Cap * 8 + 160 * 4 + 2 * kRingMaxSlots * 8 + 8 * 4 + 16 + 128;
}

template <int NW>
__global__ void __launch_bounds__((NW + 1) * 32, 1)
phase_dyn_kernel(PhaseArgs a, uint32_t m, uint32_t k, RingPlan g)
{
    constexpr int FMT = kFmtU8;
    constexpr int kThreads = (NW + 1) * 32;
    extern __shared__ __align__(128) uint8_t smem_raw[];
    const uint32_t NS = g.NS;
    const int RC = (int)g.RC, pitch = (int)g.pitch;
    uint8_t* ring0 = smem_raw;
    uint2* queues = reinterpret_cast<uint2*>(ring0 + (size_t)NS * g.slot_bytes);
    uint32_t* tbl = reinterpret_cast<uint32_t*>(queues + NW * kDynQ1Cap);
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(tbl + 160);  // full[NS], empty[NS]
    int* eoff = reinterpret_cast<int*>(bars + 2 * kRingMaxSlots);                 // e[4], f[4]
    uint32_t* next_task = reinterpret_cast<uint32_t*>(eoff + 8);
    __shared__ int delta_cta;

    const uint32_t b = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t L = a.L;
    const uint32_t cls = a.order[((size_t)b * a.order_stride + (m % a.order_stride)) * 16 + k];
    const int ci = (int)(cls >> 2), cj = (int)(cls & 3u);
    uint8_t* lat = a.lats + (size_t)b * a.lat_bytes;
    const uint32_t bar_full = smem_u32(bars), bar_empty = bar_full + 8u * NS;

    for (int q = threadIdx.x; q < kTableSize; q += kThreads)
        tbl[q] = a.tables[(size_t)b * kTableSize + q];
    if (threadIdx.x == 0) {
        delta_cta = 0;
        *next_task = 0u;
        for (uint32_t s = 0; s < NS; ++s) {
            mbar_init(bar_full + 8u * s, 1);
            mbar_init(bar_empty + 8u * s, 32);  // 16 tasks of step c-1 + 16 tasks of step c
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        // chunk 0 holds no active row of this band: only step 0 reads it
        asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0], 16;" ::"r"(bar_empty) : "memory");
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

    if (warp == NW) {
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
    } else {
        // ---------------- consumer warps ----------------
        const StepKey sk = make_step_key(a.seeds[b], a.t_begin + m, k, cls);
        uint2* q1 = queues + warp * kDynQ1Cap;
        const uint32_t lt = (1u << lane) - 1u;
        const int tmask = (1 << g.tpr_log2) - 1;
        const int wrap = ring_bytes, wrap_below = pitch;  // sites of ring row 0 take the wrapping stencil
        const uint32_t bm = 0xFFu << (8 * cj);
        // Q1 is linear, entries [0, n1); the first o1 of them belong to the previous task
        // (step s_old, whose chunks sit in slots slot_old - 1 and slot_old)
        uint32_t n1 = 0, o1 = 0, s_old = 0, slot_old = 0;
        bool has_old = false;
        int delta = 0;
        uint32_t cur_s = 0, slot = 1 % NS, par = (1 / NS) & 1u;  // slot, parity of chunk cur_s + 1

        auto grab = [&]() {
            uint32_t t = 0;
            if (lane == 0) t = atomicAdd(next_task, 1u);
            return __shfl_sync(0xFFFFFFFFu, t, 0);
        };
        // the task of step st (chunk st + 1 in slot sl) is finished: its two chunks lose a reader
        auto complete = [&](uint32_t sl) {
            if (lane == 0) {
                mbar_arrive(bar_empty + 8u * sl);
                mbar_arrive(bar_empty + 8u * (sl == 0 ? NS - 1 : sl - 1));
            }
        };
        // draw + neighbour compare, then stencil + accept + write for the lanes that go on
        auto one = [&](uint2 e) {
            uint4 v;
            if (ring_level1<FMT>(e, ring0, eoff, sk, v, wrap))
                delta += ring_level2<FMT>(v, ring0, eoff, lat, tbl, wrap, wrap_below);
        };
        // everything queued runs now (a partial batch): n1 < 32
        auto flush = [&]() {
            if ((uint32_t)lane < n1) one(q1[lane]);
            __syncwarp();
            n1 = 0;
            o1 = 0;
        };
        // full batches from the front of Q1 (two at a time while 64 wait); the leftover
        // (< 32) moves to the front.  Old entries (o1 < 32 of them) are in the first batch.
        auto run_batches = [&]() {
            if (n1 < 32u) return;
            uint32_t head = 0;
            while (n1 - head >= 64u) {
                uint4 va, vb;
                const bool ga = ring_level1<FMT>(q1[head + lane], ring0, eoff, sk, va, wrap);
                const bool gb = ring_level1<FMT>(q1[head + 32 + lane], ring0, eoff, sk, vb, wrap);
                if (ga) delta += ring_level2<FMT>(va, ring0, eoff, lat, tbl, wrap, wrap_below);
                if (gb) delta += ring_level2<FMT>(vb, ring0, eoff, lat, tbl, wrap, wrap_below);
                head += 64u;
            }
            if (n1 - head >= 32u) {
                one(q1[head + lane]);
                head += 32u;
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

        if (n_steps) mbar_wait(bar_full, 0u);  // the prologue chunk
        uint32_t gi = grab();
        while ((gi >> 4) < n_steps) {
            const uint32_t s = gi >> 4;
            const int task = (int)(gi & 15u), rho = task >> g.tpr_log2, tau = task & tmask;
            gi = grab();  // the next task's number is on its way while this one runs
            // never wait for a chunk whose load may depend on a task this warp has not finished
            if (has_old && s + 2 >= s_old + NS) {
                flush();
                complete(slot_old);
                has_old = false;
            }
            while (cur_s < s) {
                ++cur_s;
                if (++slot == NS) { slot = 0; par ^= 1u; }
            }
            // both chunks this task reads: chunk s (the rows above) and chunk s + 1.  A warp that
            // skipped steps has not seen chunk s arrive yet; neither barrier can be a phase ahead,
            // their slots are not reloaded before this task is finished.
            mbar_wait(bar_full + 8u * (slot == 0 ? NS - 1 : slot - 1), slot == 0 ? par ^ 1u : par);
            mbar_wait(bar_full + 8u * slot, par);
            const int colb = tau * kRingTaskB + 16 * lane;  // first core byte of this lane's 16
            if ((S0 + s) * g.R + (uint32_t)rho < g.n_groups) {
                const int rowoff = (int)slot * slot_bytes + 4 * rho * pitch + kRingHaloB + colb;
                const int upoff = (slot == 0 && rho == 0) ? ring_bytes - pitch : -pitch;
                const uint32_t site0 = (uint32_t)(RC * (int)(S0 + s) + 4 * rho + ci) * L + (uint32_t)(j0b + colb);
                const uint8_t* rowp = ring0 + rowoff;
                uint4 wc = make_uint4(0, 0, 0, 0), wu = wc, wd = wc;
                uint32_t pv = 0, nx = 0;
                if (colb < wb) {
                    wc = *reinterpret_cast<const uint4*>(rowp);
                    wu = *reinterpret_cast<const uint4*>(rowp + upoff);
                    wd = *reinterpret_cast<const uint4*>(rowp + pitch);
                    pv = *reinterpret_cast<const uint32_t*>(rowp - 4);
                    nx = *reinterpret_cast<const uint32_t*>(rowp + 16);
                }
                const uint32_t c4[4] = {wc.x, wc.y, wc.z, wc.w};
                const uint32_t u4[4] = {wu.x, wu.y, wu.z, wu.w};
                const uint32_t d4[4] = {wd.x, wd.y, wd.z, wd.w};
                uint32_t nb[4];
#pragma unroll
                for (int w = 0; w < 4; ++w) {
                    // word w = sites 4w..4w+3 of this lane's 16; the active one is byte cj
                    const uint32_t lw = __funnelshift_l(w == 0 ? pv : c4[w - 1], c4[w], 8);
                    const uint32_t rw = __funnelshift_r(c4[w], w == 3 ? nx : c4[w + 1], 8);
                    nb[w] = ((c4[w] ^ u4[w]) | (c4[w] ^ d4[w]) | (c4[w] ^ lw) | (c4[w] ^ rw)) & bm;  // S9
                }
                if (__any_sync(0xFFFFFFFFu, (nb[0] | nb[1] | nb[2] | nb[3]) != 0u)) {
                    const uint32_t so = (uint32_t)(rowoff + cj), si = site0 + (uint32_t)cj;
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
            }
            // sites of the previous task must be finished now (then n1 < 32)
            if (o1) flush();
            if (has_old) complete(slot_old);
            has_old = n1 != 0u;
            if (has_old) {
                s_old = s;
                slot_old = slot;
                o1 = n1;
            } else {
                complete(slot);
            }
        }
        // drain: everything left was queued by the last task
        if (n1) flush();
        if (has_old) complete(slot_old);
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
// Host side: RING's geometry (ring_plan) with DYN's fixed shared-memory part
// ---------------------------------------------------------------------------
constexpr int kDynWarps = 24;

inline bool dyn_supported(int fmt, uint32_t L)
{
    return fmt == kFmtU8 && ring_supported(fmt, L);
}

template <int NW>
inline int dyn_plan_nw(uint32_t L, uint32_t B, RingPlan* p)
{
    int smem_optin = 0;  // per call (the function attribute is per device)
    {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaFuncSetAttribute(phase_dyn_kernel<NW>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 256);
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
    while (want > 3 && want * p->slot_bytes + dyn_fixed_bytes<NW>() > (uint32_t)smem_optin - 256) --want;
    if (max_chunks < want) want = max_chunks < 3 ? 3 : max_chunks;
    p->NS = want;
    p->smem_bytes = p->NS * p->slot_bytes + dyn_fixed_bytes<NW>();
    return 0;
}

inline int dyn_warps()
{
    static int nw = 0;
    if (nw == 0) {
        nw = kDynWarps;
        if (const char* e = getenv("PGG_DYN_WARPS")) nw = atoi(e);
        if (nw != 16 && nw != 20 && nw != 24 && nw != 28) nw = kDynWarps;
    }
    return nw;
}

inline int dyn_plan(uint32_t L, uint32_t B, RingPlan* p)
{
    switch (dyn_warps()) {
    case 16: return dyn_plan_nw<16>(L, B, p);
    case 20: return dyn_plan_nw<20>(L, B, p);
    case 28: return dyn_plan_nw<28>(L, B, p);
    default: return dyn_plan_nw<24>(L, B, p);
    }
}

inline void dyn_launch(const RingPlan& p, const PhaseArgs& a, uint32_t m, uint32_t k, uint32_t B,
                       cudaStream_t stream)
{
    dim3 grid(p.n_strips * p.nb, B);
    switch (dyn_warps()) {
    case 16: phase_dyn_kernel<16><<<grid, 17 * 32, p.smem_bytes, stream>>>(a, m, k, p); break;
    case 20: phase_dyn_kernel<20><<<grid, 21 * 32, p.smem_bytes, stream>>>(a, m, k, p); break;
    case 28: phase_dyn_kernel<28><<<grid, 29 * 32, p.smem_bytes, stream>>>(a, m, k, p); break;
    default: phase_dyn_kernel<24><<<grid, 25 * 32, p.smem_bytes, stream>>>(a, m, k, p); break;
    }
}

}  // namespace pgg
