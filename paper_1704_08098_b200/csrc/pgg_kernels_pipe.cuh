// pgg_kernels_pipe.cuh -- the PIPE phase kernel (K1 uint8, K2 bit-packed): the
// TILE kernel's staging (pgg_kernels_tile.cuh) turned into a warp-specialised
// producer / consumer pipeline with no block-wide barrier in the tile loop.
//
//   * one persistent CTA per SM: 16 consumer warps + 1 producer warp;
//   * the producer warp keeps S (<= 5) tiles of 64 rows x 512 bytes (+ halo)
//     in flight with bulk-async copies (cp.async.bulk -> SASS UBLKCP) that
//     complete on a per-stage "full" mbarrier; it re-arms a stage when its
//     "empty" mbarrier has collected one arrival from each consumer warp;
//   * consumer warp w owns active row w of every tile (row 4w + ci): each lane
//     tests 4 active sites (uint8; one 16-byte shared load per lattice row) or
//     4 words = 32 active sites (bit-packed) for "all four neighbours equal
//     s_x" (S9) with word-wide logic, and the survivors are compacted into a
//     per-warp ring queue in shared memory;
//   * full batches of 32 queued sites run Philox, the neighbour compare, the
//     14-site signed stencil A_x - A_y, the threshold compare and the in-place
//     write (a3-a7).  A warp releases tile n-1 only after it has scanned tile
//     n, so a leftover (< 32 sites) is batched with the next tile's sites
//     instead of running at low lane occupancy.
#pragma once
#include "pgg_kernels_tile.cuh"

namespace pgg {

constexpr int kPipeConsumers = kTileTH / 4;            // one warp per active row of a tile
constexpr int kPipeThreads = (kPipeConsumers + 1) * 32;
constexpr int kPipeQueueCap = 512;                     // ring entries per warp (power of two)
constexpr int kPipeMaxStages = 5;
constexpr int kPipeFixedBytes = kPipeConsumers * kPipeQueueCap * 4 + 160 * 4 + 2 * kPipeMaxStages * 8 + 128;

__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// Queue entry: tile parity << 31 | stage row << 16 | site column in the staged row
__device__ __forceinline__ uint32_t pipe_entry(uint32_t par, int r, int c)
{
    return (par << 31) | ((uint32_t)r << 16) | (uint32_t)c;
}

// One tile as a consumer sees it
struct PipeTile {
    const uint8_t* smem;
    int i0;   // first core row
    int j0;   // first core SITE column
};

// Steps a3-a7 for one queued site.  Returns the change of the cooperator count.
template <int FMT>
__device__ __forceinline__ int pipe_process(uint32_t e, uint32_t par_cur, const PipeTile& cur,
                                            const PipeTile& prev, uint8_t* __restrict__ lat,
                                            uint32_t L, const StepKey& sk,
                                            const uint32_t* __restrict__ tbl)
{
    const bool is_cur = (e >> 31) == par_cur;
    const uint8_t* tile = is_cur ? cur.smem : prev.smem;
    const int i0 = is_cur ? cur.i0 : prev.i0, j0 = is_cur ? cur.j0 : prev.j0;
    const int r = (int)((e >> 16) & 0x7Fu), c = (int)(e & 0xFFFFu);
    constexpr int halo_sites = (FMT == kFmtU8) ? kTileHaloB : kTileHaloB * 8;
    const uint32_t site = (uint32_t)(i0 + r - 3) * L + (uint32_t)(j0 + c - halo_sites);
    uint32_t x0, u;
    step_draw(sk, site, x0, u);
    const uint32_t dir = x0 >> 30;  // 0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1)
    // e = unit step towards y, f = perpendicular unit step (tile-local site coords)
    const int er = dir == 0 ? -1 : dir == 1 ? 1 : 0;
    const int ec = dir == 2 ? -1 : dir == 3 ? 1 : 0;
    const int fr = dir < 2 ? 0 : 1, fc = dir < 2 ? 1 : 0;
    int sx, sy, dA;
    if (FMT == kFmtU8) {
        const uint8_t* p = tile + r * kTilePitch + c;
        const int eo = er * kTilePitch + ec, fo = fr * kTilePitch + fc;
        sx = p[0];
        sy = p[eo];
        if (sx == sy) return 0;
        // A_x - A_y with A = 5 s + 2 (nearest + diagonal) + axial distance-2 (include/pgg.h):
        // weights of x's 13-site stencil minus those of y's, at offset (a along e, b along f)
        dA = p[-2 * eo] + p[-eo] - p[2 * eo] - p[3 * eo] + 3 * (sx - sy)
           + 2 * (p[-eo + fo] + p[-eo - fo] - p[2 * eo + fo] - p[2 * eo - fo])
           + p[2 * fo] + p[-2 * fo] - p[eo + 2 * fo] - p[eo - 2 * fo];
    } else {
        auto S = [&](int a, int b) { return tile_get<kFmtBits>(tile, r + a * er + b * fr, c + a * ec + b * fc); };
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
__global__ void __launch_bounds__(kPipeThreads, 1)
phase_pipe_kernel(PhaseArgs a, uint32_t m, uint32_t k, TilePlan g)
{
    extern __shared__ __align__(128) uint8_t smem_raw[];
    uint8_t* stages = smem_raw;
    uint32_t* queues = reinterpret_cast<uint32_t*>(smem_raw + (size_t)g.stages * kTileStageBytes);
    uint32_t* tbl = queues + kPipeConsumers * kPipeQueueCap;
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(tbl + 160);  // full[S], empty[S]
    __shared__ int delta_cta;

    const uint32_t b = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t L = a.L;
    const uint32_t cls = a.order[((size_t)b * a.order_stride + (m % a.order_stride)) * 16 + k];
    const int ci = (int)(cls >> 2), cj = (int)(cls & 3u);
    uint8_t* lat = a.lats + (size_t)b * a.lat_bytes;
    const uint32_t S = g.stages;

    for (int q = threadIdx.x; q < kTableSize; q += kPipeThreads)
        tbl[q] = a.tables[(size_t)b * kTableSize + q];
    if (threadIdx.x == 0) {
        delta_cta = 0;
        for (uint32_t s = 0; s < S; ++s) {
            mbar_init(smem_u32(&bars[s]), 1);
            mbar_init(smem_u32(&bars[S + s]), kPipeConsumers);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const uint32_t G = gridDim.x;
    const uint32_t n_my = blockIdx.x < g.n_tiles ? (g.n_tiles - blockIdx.x + G - 1) / G : 0;
    const uint32_t stage0 = smem_u32(stages);

    if (warp == kPipeConsumers) {
        // ---------------- producer warp ----------------
        for (uint32_t n = 0; n < n_my; ++n) {
            const uint32_t st = n % S;
            if (n >= S) mbar_wait(smem_u32(&bars[S + st]), ((n / S) - 1u) & 1u);
            const TileCoord t = tile_coord(g, L, blockIdx.x + n * G);
            tile_issue(lat, g, L, t, stage0 + st * kTileStageBytes, smem_u32(&bars[st]), lane);
        }
    } else {
        // ---------------- consumer warps ----------------
        const StepKey sk = make_step_key(a.seeds[b], a.t_begin + m, k, cls);
        uint32_t* q = queues + warp * kPipeQueueCap;
        constexpr uint32_t qmask = kPipeQueueCap - 1;
        const uint32_t lt = (1u << lane) - 1u;
        uint32_t head = 0, tail = 0, prev_tail = 0;
        PipeTile cur{nullptr, 0, 0}, prev{nullptr, 0, 0};
        int delta = 0;

        for (uint32_t n = 0; n < n_my; ++n) {
            const uint32_t st = n % S, par = n & 1u;
            const TileCoord t = tile_coord(g, L, blockIdx.x + n * G);
            cur.smem = stages + (size_t)st * kTileStageBytes;
            cur.i0 = t.i0;
            cur.j0 = (FMT == kFmtU8) ? t.j0b : t.j0b * 8;
            mbar_wait(smem_u32(&bars[st]), (n / S) & 1u);

            if (4 * warp < t.th) {
                const int r = 3 + ci + 4 * warp;
                const bool in = 16 * lane < t.twb;
                const uint8_t* rowp = cur.smem + r * kTilePitch + kTileHaloB + 16 * lane;
                uint4 wc = make_uint4(0, 0, 0, 0), wu = wc, wd = wc;
                uint32_t pv = 0, nx = 0;
                if (in) {
                    wc = *reinterpret_cast<const uint4*>(rowp);
                    wu = *reinterpret_cast<const uint4*>(rowp - kTilePitch);
                    wd = *reinterpret_cast<const uint4*>(rowp + kTilePitch);
                    pv = *reinterpret_cast<const uint32_t*>(rowp - 4);
                    nx = *reinterpret_cast<const uint32_t*>(rowp + 16);
                }
                const uint32_t c4[4] = {wc.x, wc.y, wc.z, wc.w};
                const uint32_t u4[4] = {wu.x, wu.y, wu.z, wu.w};
                const uint32_t d4[4] = {wd.x, wd.y, wd.z, wd.w};
                if (FMT == kFmtU8) {
                    // word q = sites 4q..4q+3 of this lane's 16; the active one is byte cj
                    const uint32_t bm = 0xFFu << (8 * cj);
#pragma unroll
                    for (int w = 0; w < 4; ++w) {
                        const uint32_t lw = __funnelshift_l(w == 0 ? pv : c4[w - 1], c4[w], 8);
                        const uint32_t rw = __funnelshift_r(c4[w], w == 3 ? nx : c4[w + 1], 8);
                        const uint32_t nb = ((c4[w] ^ u4[w]) | (c4[w] ^ d4[w]) | (c4[w] ^ lw) | (c4[w] ^ rw)) & bm;  // S9
                        const bool pred = in && nb != 0u;
                        const uint32_t mk = __ballot_sync(0xFFFFFFFFu, pred);
                        if (pred)
                            q[(tail + __popc(mk & lt)) & qmask] =
                                pipe_entry(par, r, kTileHaloB + 16 * lane + 4 * w + cj);
                        tail += __popc(mk);
                    }
                    __syncwarp();
                    while (tail - head >= 32u) {
                        delta += pipe_process<FMT>(q[(head + lane) & qmask], par, cur, prev, lat, L, sk, tbl);
                        head += 32u;
                    }
                } else {
                    // word w = 32 sites; the 8 active ones are bits cj + 4 b
                    const uint32_t cm = 0x11111111u << cj;
#pragma unroll
                    for (int w = 0; w < 4; ++w) {
                        const uint32_t lw = __funnelshift_l(w == 0 ? pv : c4[w - 1], c4[w], 1);
                        const uint32_t rw = __funnelshift_r(c4[w], w == 3 ? nx : c4[w + 1], 1);
                        const uint32_t nb = ((c4[w] ^ u4[w]) | (c4[w] ^ d4[w]) | (c4[w] ^ lw) | (c4[w] ^ rw)) & cm;  // S9
                        if (__any_sync(0xFFFFFFFFu, nb != 0u)) {
#pragma unroll
                            for (int bb = 0; bb < 8; ++bb) {
                                const int bit = cj + 4 * bb;
                                const bool pred = (nb >> bit) & 1u;
                                const uint32_t mk = __ballot_sync(0xFFFFFFFFu, pred);
                                if (pred)
                                    q[(tail + __popc(mk & lt)) & qmask] =
                                        pipe_entry(par, r, 8 * (kTileHaloB + 16 * lane + 4 * w) + bit);
                                tail += __popc(mk);
                            }
                            __syncwarp();
                            while (tail - head >= 32u) {
                                delta += pipe_process<FMT>(q[(head + lane) & qmask], par, cur, prev, lat, L, sk, tbl);
                                head += 32u;
                            }
                        }
                    }
                }
            }
            // sites of tile n-1 still queued (then fewer than 32 are queued in all): flush them
            if (head != prev_tail && (int32_t)(prev_tail - head) > 0) {
                const uint32_t cnt = tail - head;
                if ((uint32_t)lane < cnt)
                    delta += pipe_process<FMT>(q[(head + lane) & qmask], par, cur, prev, lat, L, sk, tbl);
                head = tail;
            }
            __syncwarp();
            if (n > 0 && lane == 0) mbar_arrive(smem_u32(&bars[S + (n - 1u) % S]));  // tile n-1 is free
            prev = cur;
            prev_tail = tail;
        }
        // drain (all remaining sites belong to the last tile)
        {
            const uint32_t cnt = tail - head;
            if ((uint32_t)lane < cnt)
                delta += pipe_process<FMT>(q[(head + lane) & qmask], (n_my - 1u) & 1u, prev, prev, lat, L, sk, tbl);
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
inline int pipe_plan(int fmt, uint32_t L, uint32_t B, TilePlan* p)
{
    int sm_count = 0, smem_optin = 0;  // per call: the function attribute is per device, and a plan costs nothing next to 16 n_mcs launches
    {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (e != cudaSuccess) return (int)e;
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaFuncSetAttribute(phase_pipe_kernel<kFmtU8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 1024);
        if (e != cudaSuccess) return (int)e;
        e = cudaFuncSetAttribute(phase_pipe_kernel<kFmtBits>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 1024);
        if (e != cudaSuccess) return (int)e;
        sm_count = sms;
    }
    p->row_bytes = fmt == kFmtU8 ? L : L / 8;
    p->n_strips = (p->row_bytes + kTileTWB - 1) / kTileTWB;
    p->n_rowblocks = (L + kTileTH - 1) / kTileTH;
    p->n_tiles = p->n_strips * p->n_rowblocks;
    uint32_t want_stages = kPipeMaxStages;
    if (const char* e = getenv("PGG_PIPE_STAGES")) want_stages = (uint32_t)atoi(e);
    if (want_stages > (uint32_t)kPipeMaxStages) want_stages = kPipeMaxStages;
    if (want_stages < 2) want_stages = 2;
    while (kPipeFixedBytes + want_stages * kTileStageBytes > (uint32_t)smem_optin - 1024) --want_stages;
    uint32_t ctas = (uint32_t)sm_count;
    uint32_t gx = p->n_tiles < ctas ? p->n_tiles : ctas;
    if (B > 1) {  // share the machine between lattices
        uint32_t per_lat = (ctas + B - 1) / B;
        if (gx > per_lat) gx = per_lat;
    }
    const uint32_t per = (p->n_tiles + gx - 1) / gx;
    uint32_t stages = want_stages;
    if (per + 1 < stages) stages = per + 1 < 2 ? 2 : per + 1;
    p->stages = stages;
    p->grid_x = gx;
    p->smem_bytes = kPipeFixedBytes + stages * kTileStageBytes;
    return 0;
}

inline void pipe_launch(const TilePlan& p, int fmt, const PhaseArgs& a, uint32_t m, uint32_t k,
                        uint32_t B, cudaStream_t stream)
{
    dim3 grid(p.grid_x, B);
    if (fmt == kFmtU8)
        phase_pipe_kernel<kFmtU8><<<grid, kPipeThreads, p.smem_bytes, stream>>>(a, m, k, p);
    else
        phase_pipe_kernel<kFmtBits><<<grid, kPipeThreads, p.smem_bytes, stream>>>(a, m, k, p);
}

}  // namespace pgg
