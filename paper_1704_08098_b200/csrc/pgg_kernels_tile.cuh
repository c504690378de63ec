// pgg_kernels_tile.cuh -- the TILE phase kernel (K1 uint8, K2 bit-packed).
//
// One launch = one phase (one sublattice class) over B lattices.  Persistent
// CTAs walk over tiles of TH rows x TWB bytes.  Each tile plus its halo (3 rows
// above and below, 16 bytes left and right -- 3 sites are needed, 16 bytes keep
// every copy 16-byte aligned) is staged into shared memory by bulk-async copies
// (cp.async.bulk, SASS UBLKCP: the TMA engine's 1-D path) that complete on an
// mbarrier, S stages deep, so HBM requests stay in flight while warps compute.
// Periodic wrap is resolved per row / per halo chunk on the
// source address; TMA tensor maps zero-fill out of bounds and cannot wrap.
//
// Compute (steps a3-a8): each lane tests one active site (uint8)
// or one 32-site word = 8 active sites (bits) for "all four neighbours equal
// s_x" (S9: no draw can change such a site).  Surviving sites are compacted
// through a per-warp shared-memory queue; full batches of 32 then run Philox,
// and those whose neighbour differs evaluate the 14-site signed stencil
// A_x - A_y from the tile, look up the threshold and flip in global memory.
// In-place writes are race-free (S1): nothing within Manhattan distance 3 of
// an active site is written in the same phase.
#pragma once
#include <cstdlib>

#include "pgg_common.cuh"

namespace pgg {

constexpr int kTileTH = 64;    // core rows per tile
constexpr int kTileTWB = 512;  // core bytes per tile row (512 sites u8, 4096 sites bits)
constexpr int kTileHaloB = 16; // halo bytes left / right
constexpr int kTileRows = kTileTH + 6;
constexpr int kTilePitch = kTileTWB + 2 * kTileHaloB;
constexpr int kTileStageBytes = kTileRows * kTilePitch;
constexpr int kTileWarps = 8;
constexpr int kTileThreads = kTileWarps * 32;
constexpr int kTileQueueCap = 32 + 256;  // entries per warp (bits: one round adds up to 256)
constexpr int kTileMaxStages = 5;

struct TilePlan {
    uint32_t row_bytes;    // bytes per lattice row
    uint32_t n_strips;     // tiles across
    uint32_t n_rowblocks;  // tiles down
    uint32_t n_tiles;      // per lattice
    uint32_t stages;
    uint32_t grid_x;       // persistent CTAs per lattice
    uint32_t smem_bytes;
};

inline bool tile_supported(int fmt, uint32_t L)
{
    if (L > 32768) return false;  // tile-local coordinates are packed into 16 bits
    return fmt == kFmtU8 ? (L % 16 == 0) : (L % 128 == 0);
}

// ---------------------------------------------------------------------------
// mbarrier / bulk-copy primitives (PTX; sm_90+ forms, native on sm_100a)
// ---------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
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
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
        "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}

// ---------------------------------------------------------------------------
// Tile geometry of one CTA iteration
// ---------------------------------------------------------------------------
struct TileCoord {
    int i0;   // first core row
    int j0b;  // first core byte within the row
    int th;   // core rows (multiple of 4)
    int twb;  // core bytes (multiple of 16)
};

__device__ __forceinline__ TileCoord tile_coord(const TilePlan& g, uint32_t L, uint32_t id)
{
    // vertical-major order: CTAs that run side by side hold vertically adjacent
    // tiles, so the shared halo rows are fetched from DRAM once and hit L2 after
    const uint32_t strip = id / g.n_rowblocks, rb = id - strip * g.n_rowblocks;
    TileCoord t;
    t.i0 = (int)(rb * kTileTH);
    t.j0b = (int)(strip * kTileTWB);
    t.th = min(kTileTH, (int)L - t.i0);
    t.twb = min(kTileTWB, (int)g.row_bytes - t.j0b);
    return t;
}

// Issued by one warp: stage the tile and its halo.  Row r of the stage holds
// lattice row (i0 - 3 + r) mod L, bytes [j0b - 16, j0b + twb + 16) mod row_bytes.
__device__ __forceinline__ void tile_issue(const uint8_t* __restrict__ lat, const TilePlan& g,
                                           uint32_t L, const TileCoord& t, uint32_t stage_smem,
                                           uint32_t bar, int lane)
{
    const int rows = t.th + 6;
    const int rb = (int)g.row_bytes;
    if (lane == 0) mbar_expect_tx(bar, (uint32_t)(rows * (t.twb + 2 * kTileHaloB)));
    __syncwarp();
    const bool interior = (t.j0b >= kTileHaloB) && (t.j0b + t.twb + kTileHaloB <= rb);
    const int jl = t.j0b >= kTileHaloB ? t.j0b - kTileHaloB : rb - kTileHaloB;
    const int jr = t.j0b + t.twb < rb ? t.j0b + t.twb : 0;
    for (int r = lane; r < rows; r += 32) {
        int gi = t.i0 - 3 + r;
        gi = gi < 0 ? gi + (int)L : gi;
        gi = gi >= (int)L ? gi - (int)L : gi;
        const uint8_t* src = lat + (size_t)gi * (size_t)rb;
        const uint32_t dst = stage_smem + (uint32_t)(r * kTilePitch);
        if (interior) {
            bulk_g2s(dst, src + jl, (uint32_t)(t.twb + 2 * kTileHaloB), bar);
        } else {
            bulk_g2s(dst, src + jl, kTileHaloB, bar);
            bulk_g2s(dst + kTileHaloB, src + t.j0b, (uint32_t)t.twb, bar);
            bulk_g2s(dst + kTileHaloB + (uint32_t)t.twb, src + jr, kTileHaloB, bar);
        }
    }
}

// ---------------------------------------------------------------------------
// Site access inside a staged tile.  (r, c) are tile-local SITE coordinates:
// r = stage row, c = site column counted from the first staged byte.
// ---------------------------------------------------------------------------
template <int FMT>
__device__ __forceinline__ int tile_get(const uint8_t* tile, int r, int c);

template <>
__device__ __forceinline__ int tile_get<kFmtU8>(const uint8_t* tile, int r, int c)
{
    return tile[r * kTilePitch + c];
}
template <>
__device__ __forceinline__ int tile_get<kFmtBits>(const uint8_t* tile, int r, int c)
{
    return (tile[r * kTilePitch + (c >> 3)] >> (c & 7)) & 1;
}

// Queue entry: sx<<31 | up<<30 | dn<<29 | lf<<28 | rt<<27 | r<<16 | c
__device__ __forceinline__ uint32_t make_entry(int sx, int up, int dn, int lf, int rt, int r, int c)
{
    return ((uint32_t)sx << 31) | ((uint32_t)up << 30) | ((uint32_t)dn << 29) |
           ((uint32_t)lf << 28) | ((uint32_t)rt << 27) | ((uint32_t)r << 16) | (uint32_t)c;
}

// Steps a3-a7 for one compacted site.  Returns the change of the cooperator count.
template <int FMT>
__device__ __forceinline__ int tile_process_entry(uint32_t e, const uint8_t* __restrict__ tile,
                                                  const TileCoord& t, uint8_t* __restrict__ lat,
                                                  uint32_t L, const StepKey& sk,
                                                  const uint32_t* __restrict__ tbl)
{
    const int r = (int)((e >> 16) & 0x7FFu), c = (int)(e & 0xFFFFu);
    const int sx = (int)(e >> 31);
    const int halo_sites = (FMT == kFmtU8) ? kTileHaloB : kTileHaloB * 8;
    const int j0 = (FMT == kFmtU8) ? t.j0b : t.j0b * 8;
    const uint32_t gi = (uint32_t)(t.i0 + r - 3), gj = (uint32_t)(j0 + c - halo_sites);
    const uint32_t site = gi * L + gj;
    uint32_t x0, u;
    step_draw(sk, site, x0, u);
    const uint32_t dir = x0 >> 30;  // 0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1)
    const int sy = (int)((e >> (30u - dir)) & 1u);
    if (sy == sx) return 0;
    // e = unit step towards y, f = perpendicular unit step (tile-local site coords)
    const int er = dir == 0 ? -1 : dir == 1 ? 1 : 0;
    const int ec = dir == 2 ? -1 : dir == 3 ? 1 : 0;
    const int fr = dir < 2 ? 0 : 1, fc = dir < 2 ? 1 : 0;
    auto S = [&](int a, int b) { return tile_get<FMT>(tile, r + a * er + b * fr, c + a * ec + b * fc); };
    // A_x - A_y, with A = 5 s + 2 (nearest + diagonal) + axial distance-2 (include/pgg.h):
    // the weights of x's 13-site stencil minus those of y's, at offset (a along e, b along f)
    const int dA = S(-2, 0) + S(-1, 0) + 3 * (sx - sy) - S(2, 0) - S(3, 0)
                 + 2 * (S(-1, 1) + S(-1, -1) - S(2, 1) - S(2, -1))
                 + S(0, 2) + S(0, -2) - S(1, 2) - S(1, -2);
    const uint32_t T = tbl[table_index(dA, sx - sy)];
    if (u < T) {
        if (FMT == kFmtU8) {
            lat[site] = (uint8_t)sy;
        } else {
            atomicXor(reinterpret_cast<uint32_t*>(lat) + (site >> 5), 1u << (site & 31u));
        }
        return sy - sx;
    }
    return 0;
}

template <int FMT>
__global__ void __launch_bounds__(kTileThreads)
phase_tile_kernel(PhaseArgs a, uint32_t m, uint32_t k, TilePlan g)
{
    extern __shared__ __align__(128) uint8_t smem_raw[];
    uint8_t* stages = smem_raw;
    uint32_t* queues = reinterpret_cast<uint32_t*>(smem_raw + (size_t)g.stages * kTileStageBytes);
    uint32_t* tbl = queues + kTileWarps * kTileQueueCap;
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(tbl + 160);
    __shared__ int delta_part[kTileWarps];

    const uint32_t b = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t L = a.L;
    const uint32_t cls = a.order[((size_t)b * a.order_stride + (m % a.order_stride)) * 16 + k];
    const int ci = (int)(cls >> 2), cj = (int)(cls & 3u);
    const StepKey sk = make_step_key(a.seeds[b], a.t_begin + m, k, cls);
    uint8_t* lat = a.lats + (size_t)b * a.lat_bytes;

    for (int q = threadIdx.x; q < kTableSize; q += kTileThreads)
        tbl[q] = a.tables[(size_t)b * kTableSize + q];
    if (threadIdx.x == 0) {
        for (uint32_t s = 0; s < g.stages; ++s) mbar_init(smem_u32(&bars[s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const uint32_t G = gridDim.x;
    const uint32_t n_my = blockIdx.x < g.n_tiles ? (g.n_tiles - blockIdx.x + G - 1) / G : 0;
    const uint32_t S = g.stages;
    const uint32_t stage0 = smem_u32(stages);

    // prologue: S-1 tiles in flight
    if (warp == 0) {
        for (uint32_t n = 0; n + 1 < S && n < n_my; ++n) {
            const TileCoord t = tile_coord(g, L, blockIdx.x + n * G);
            tile_issue(lat, g, L, t, stage0 + n * kTileStageBytes, smem_u32(&bars[n]), lane);
        }
    }

    uint32_t* q = queues + warp * kTileQueueCap;
    int delta = 0;

    for (uint32_t n = 0; n < n_my; ++n) {
        // every warp is done with the stage tile n-1 lived in: refill it with tile n+S-1
        __syncthreads();
        if (warp == 0 && n + S - 1 < n_my) {
            const uint32_t nn = n + S - 1, st = nn % S;
            const TileCoord t = tile_coord(g, L, blockIdx.x + nn * G);
            tile_issue(lat, g, L, t, stage0 + st * kTileStageBytes, smem_u32(&bars[st]), lane);
        }
        const uint32_t st = n % S;
        const TileCoord t = tile_coord(g, L, blockIdx.x + n * G);
        mbar_wait(smem_u32(&bars[st]), (n / S) & 1u);
        const uint8_t* tile = stages + (size_t)st * kTileStageBytes;

        int qn = 0;  // queue fill (warp-uniform)
        const int na = t.th >> 2;
        if (FMT == kFmtU8) {
            const int nb = t.twb >> 2;  // active sites per core row
            const int nseg = (nb + 31) >> 5;
            for (int task = warp; task < na * nseg; task += kTileWarps) {
                const int ar = task / nseg, seg = task - ar * nseg;
                const int bcol = seg * 32 + lane;
                const int r = 3 + ci + 4 * ar, c = kTileHaloB + cj + 4 * bcol;
                bool nonbulk = false;
                uint32_t e = 0;
                if (bcol < nb) {
                    const uint8_t* p = tile + r * kTilePitch + c;
                    const int sx = p[0], up = p[-kTilePitch], dn = p[kTilePitch], lf = p[-1], rt = p[1];
                    nonbulk = (up + dn + lf + rt) != 4 * sx;  // S9
                    e = make_entry(sx, up, dn, lf, rt, r, c);
                }
                const uint32_t mask = __ballot_sync(0xFFFFFFFFu, nonbulk);
                if (mask) {
                    if (nonbulk) q[qn + __popc(mask & ((1u << lane) - 1u))] = e;
                    qn += __popc(mask);
                    __syncwarp();
                    if (qn >= 32) {
                        qn -= 32;
                        delta += tile_process_entry<FMT>(q[qn + lane], tile, t, lat, L, sk, tbl);
                        __syncwarp();
                    }
                }
            }
        } else {
            // bits: lane owns one 32-site word = 8 active sites (bit cj + 4q)
            const int nw = t.twb >> 2;  // core words per row
            const int nseg = (nw + 31) >> 5;
            const uint32_t clsmask = 0x11111111u << cj;
            for (int task = warp; task < na * nseg; task += kTileWarps) {
                const int ar = task / nseg, seg = task - ar * nseg;
                const int wcol = seg * 32 + lane;
                const int r = 3 + ci + 4 * ar;
                uint32_t nbm = 0, wc = 0, wu = 0, wd = 0, wl = 0, wr = 0;
                if (wcol < nw) {
                    const uint32_t* p = reinterpret_cast<const uint32_t*>(tile + r * kTilePitch + kTileHaloB) + wcol;
                    wc = p[0];
                    wu = p[-(kTilePitch / 4)];
                    wd = p[kTilePitch / 4];
                    wl = (wc << 1) | (p[-1] >> 31);   // bit q = left neighbour of site q
                    wr = (wc >> 1) | (p[1] << 31);    // bit q = right neighbour of site q
                    nbm = ((wc ^ wu) | (wc ^ wd) | (wc ^ wl) | (wc ^ wr)) & clsmask;  // S9
                }
                const int cnt = __popc(nbm);
                // exclusive prefix of cnt over the warp
                int pre = cnt;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const int v = __shfl_up_sync(0xFFFFFFFFu, pre, d);
                    if (lane >= d) pre += v;
                }
                const int total = __shfl_sync(0xFFFFFFFFu, pre, 31);
                if (total) {
                    int pos = qn + pre - cnt;
                    while (nbm) {
                        const int bit = __ffs(nbm) - 1;
                        nbm &= nbm - 1;
                        const int c = kTileHaloB * 8 + wcol * 32 + bit;
                        q[pos++] = make_entry((wc >> bit) & 1, (wu >> bit) & 1, (wd >> bit) & 1,
                                              (wl >> bit) & 1, (wr >> bit) & 1, r, c);
                    }
                    qn += total;
                    __syncwarp();
                    while (qn >= 32) {
                        qn -= 32;
                        delta += tile_process_entry<FMT>(q[qn + lane], tile, t, lat, L, sk, tbl);
                        __syncwarp();
                    }
                }
            }
        }
        // drain: the queue refers to this tile's staging buffer
        if (qn > 0) {
            if (lane < qn) delta += tile_process_entry<FMT>(q[lane], tile, t, lat, L, sk, tbl);
            __syncwarp();
        }
    }

    if (a.deltas != nullptr) {
        delta = __reduce_add_sync(0xFFFFFFFFu, delta);
        if (lane == 0) delta_part[warp] = delta;
        __syncthreads();
        if (threadIdx.x == 0) {
            int s = 0;
            for (int w = 0; w < kTileWarps; ++w) s += delta_part[w];
            if (s != 0)
                atomicAdd(a.deltas + (size_t)b * a.n_mcs + m, (unsigned long long)(long long)s);
        }
    }
}

// ---------------------------------------------------------------------------
// Host side
// ---------------------------------------------------------------------------
inline int tile_plan(int fmt, uint32_t L, uint32_t B, TilePlan* p)
{
    int sm_count = 0, smem_optin = 0;  // per call: the function attribute is per device, and a plan costs nothing next to 16 n_mcs launches
    {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaFuncSetAttribute(phase_tile_kernel<kFmtU8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 1024);
        if (e != cudaSuccess) return (int)e;
        e = cudaFuncSetAttribute(phase_tile_kernel<kFmtBits>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin - 1024);
        if (e != cudaSuccess) return (int)e;
        cudaFuncSetAttribute(phase_tile_kernel<kFmtU8>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        cudaFuncSetAttribute(phase_tile_kernel<kFmtBits>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    }
    p->row_bytes = fmt == kFmtU8 ? L : L / 8;
    p->n_strips = (p->row_bytes + kTileTWB - 1) / kTileTWB;
    p->n_rowblocks = (L + kTileTH - 1) / kTileTH;
    p->n_tiles = p->n_strips * p->n_rowblocks;
    const uint32_t fixed = kTileWarps * kTileQueueCap * 4 + 160 * 4 + kTileMaxStages * 8 + 128;
    // CTAs per SM and stages per CTA: as many stages as fit beside `cps` CTAs (>= 2).
    // PGG_TILE_CTAS_PER_SM / PGG_TILE_STAGES override the defaults (tuning knobs).
    uint32_t cps = 2, want_stages = 3;
    if (const char* e = getenv("PGG_TILE_CTAS_PER_SM")) cps = (uint32_t)atoi(e);
    if (const char* e = getenv("PGG_TILE_STAGES")) want_stages = (uint32_t)atoi(e);
    if (cps < 1) cps = 1;
    if (want_stages > (uint32_t)kTileMaxStages) want_stages = kTileMaxStages;
    uint32_t stages = 2;
    const uint32_t per_cta = (uint32_t)(228 * 1024 / cps) - 1024 - 128;
    while (stages < want_stages && fixed + (stages + 1) * kTileStageBytes <= per_cta) ++stages;
    uint32_t ctas = cps * (uint32_t)sm_count;
    uint32_t gx = p->n_tiles < ctas ? p->n_tiles : ctas;
    if (B > 1) {  // share the machine between lattices
        uint32_t per_lat = (ctas + B - 1) / B;
        if (per_lat < 1) per_lat = 1;
        if (gx > per_lat) gx = per_lat;
    }
    const uint32_t per = (p->n_tiles + gx - 1) / gx;
    if (per < stages) stages = per < 2 ? 2 : per;
    p->stages = stages;
    p->grid_x = gx;
    p->smem_bytes = fixed + stages * kTileStageBytes;
    return 0;
}

inline void tile_launch(const TilePlan& p, int fmt, const PhaseArgs& a, uint32_t m, uint32_t k,
                        uint32_t B, cudaStream_t stream)
{
    dim3 grid(p.grid_x, B);
    if (fmt == kFmtU8)
        phase_tile_kernel<kFmtU8><<<grid, kTileThreads, p.smem_bytes, stream>>>(a, m, k, p);
    else
        phase_tile_kernel<kFmtBits><<<grid, kTileThreads, p.smem_bytes, stream>>>(a, m, k, p);
}

}  // namespace pgg
