// pgg.cu -- the C ABI of libpgg (include/pgg.h): argument validation, the host
// acceptance-table builder, stream-ordered temporaries and the launch sequence
// of a sweep.  Every step of the method itself runs in the CUDA kernels.
// Compile: nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo (see build.py).
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/pgg.h"
#include "pgg_common.cuh"
#include "pgg_kernels_v0.cuh"
#include "pgg_kernels_tile.cuh"
#include "pgg_kernels_pipe.cuh"
#include "pgg_kernels_band.cuh"
#include "pgg_kernels_ring.cuh"
#include "pgg_kernels_split.cuh"
#include "pgg_kernels_dyn.cuh"
#include "pgg_kernels_resident.cuh"
#include "pgg_kernels_lean.cuh"
#include "pgg_kernels_cluster.cuh"
#include "pgg_kernels_dtile.cuh"
#include "pgg_kernels_probe.cuh"

namespace {

thread_local std::string g_last_error;
thread_local int g_variant_used = PGG_VARIANT_AUTO;
std::atomic<int> g_variant{PGG_VARIANT_AUTO};
std::atomic<unsigned long long> g_launches{0};

int32_t fail(int32_t code, const char* fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_last_error = buf;
    return code;
}

#define PGG_CUDA(call)                                                                         \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess)                                                                 \
            return fail(PGG_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_),  \
                        __FILE__, __LINE__);                                                   \
    } while (0)

#define PGG_LAUNCHED()                                                                         \
    do {                                                                                       \
        g_launches.fetch_add(1, std::memory_order_relaxed);                                    \
        PGG_CUDA(cudaGetLastError());                                                          \
    } while (0)

int32_t check_lattice_args(const void* d_lat, int32_t fmt, uint32_t L)
{
    if (d_lat == nullptr) return fail(PGG_ERR_NULL, "lattice pointer is NULL");
    if (fmt != PGG_FMT_U8 && fmt != PGG_FMT_BITS) return fail(PGG_ERR_UNSUPPORTED, "unknown fmt %d", fmt);
    if (L < 4 || L % 4 != 0 || L >= 65536)  // site indices (Philox counter word, uint32) need L*L <= 2^32 - 1
        return fail(PGG_ERR_BAD_L, "L = %u: need 4 <= L <= 65532 and L %% 4 == 0", L);
    if (fmt == PGG_FMT_BITS && L % 32 != 0)
        return fail(PGG_ERR_BAD_L, "L = %u: the bit-packed layout needs L %% 32 == 0", L);
    if ((reinterpret_cast<uintptr_t>(d_lat) & 15u) != 0)
        return fail(PGG_ERR_ALIGN, "lattice pointer must be 16-byte aligned");
    return PGG_OK;
}

inline unsigned long long lattice_bytes(int32_t fmt, uint32_t L)
{
    const unsigned long long n = (unsigned long long)L * L;
    return fmt == PGG_FMT_U8 ? n : n / 8;
}

// The library's own stream-ordered memory pool, one per device, created on first use.  Its release
// threshold is unlimited: what a call frees stays in the pool for the next call instead of going back
// to the driver at the next synchronisation (the default pool does that, and a call that needs a 32 MiB
// working copy would then pay a fresh allocation every time).  pgg_trim_workspace() gives it back.
constexpr int kMaxDevices = 64;
std::mutex g_pool_mutex;
cudaMemPool_t g_pool[kMaxDevices] = {};

cudaError_t workspace_pool(cudaMemPool_t* out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    if (g_pool[dev] == nullptr) {
        cudaMemPoolProps props{};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        e = cudaMemPoolCreate(&pool, &props);
        if (e != cudaSuccess) return e;
        unsigned long long keep = ~0ull;
        e = cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        if (e != cudaSuccess) return e;
        g_pool[dev] = pool;
    }
    *out = g_pool[dev];
    return cudaSuccess;
}

// Device temporaries of one call, returned to the stream-ordered pool on scope exit.
struct Scratch {
    cudaStream_t stream;
    std::vector<void*> ptrs;
    explicit Scratch(cudaStream_t s) : stream(s) {}
    ~Scratch()
    {
        for (void* p : ptrs) cudaFreeAsync(p, stream);
    }
    cudaError_t alloc(void** p, size_t bytes)
    {
        cudaMemPool_t pool = nullptr;
        cudaError_t e = workspace_pool(&pool);
        if (e != cudaSuccess) return e;
        e = cudaMallocFromPoolAsync(p, bytes ? bytes : 16, pool, stream);
        if (e == cudaSuccess) ptrs.push_back(*p);
        return e;
    }
};

// seeds (and, if h_tables != nullptr, acceptance tables) of B lattices -> device arrays, as kernel arguments
int32_t upload_params(uint32_t B, const uint64_t* h_seeds, const uint32_t* h_tables, uint64_t* d_seeds,
                      uint32_t* d_tables, cudaStream_t stream)
{
    for (uint32_t first = 0; first < B; first += pgg::kParamPackLattices) {
        pgg::ParamPack p;
        p.n = std::min<uint32_t>(pgg::kParamPackLattices, B - first);
        p.with_tables = h_tables != nullptr ? 1u : 0u;
        for (uint32_t a = 0; a < p.n; ++a) p.seeds[a] = h_seeds[first + a];
        if (h_tables != nullptr)
            std::memcpy(p.tables, h_tables + (size_t)first * pgg::kTableSize, sizeof(uint32_t) * p.n * pgg::kTableSize);
        pgg::upload_params_kernel<<<1, 256, 0, stream>>>(p, first, d_seeds, d_tables);
        PGG_LAUNCHED();
    }
    return PGG_OK;
}

int32_t launch_init(uint8_t* d_lats, int32_t fmt, uint32_t B, uint32_t L, double rho0,
                    const uint64_t* d_seeds, cudaStream_t stream)
{
    // thr = floor(rho0 * 2^32) in [0, 2^32]  (D4)
    const unsigned long long thr = (unsigned long long)std::floor(rho0 * 4294967296.0);
    const uint32_t n_sites = L * L;  // L <= 65532 (check_lattice_args)
    const unsigned long long lb = lattice_bytes(fmt, L);
    const uint32_t n_items = fmt == PGG_FMT_U8 ? n_sites >> 4 : n_sites >> 5;
    uint32_t gx = (n_items + 255) / 256;
    if (gx == 0) gx = 1;
    if (gx > 148u * 64u) gx = 148u * 64u;
    dim3 grid(gx, B);
    if (fmt == PGG_FMT_U8)
        pgg::init_u8_kernel<<<grid, 256, 0, stream>>>(d_lats, lb, d_seeds, n_sites, thr);
    else
        pgg::init_bits_kernel<<<grid, 256, 0, stream>>>(d_lats, lb, d_seeds, n_sites, thr);
    PGG_LAUNCHED();
    return PGG_OK;
}

int32_t launch_density(const uint8_t* d_lats, int32_t fmt, uint32_t B, uint32_t L,
                       unsigned long long* d_out, uint32_t out_stride, cudaStream_t stream)
{
    const unsigned long long lb = lattice_bytes(fmt, L);
    unsigned long long n16 = lb >> 4;
    uint32_t gx = (uint32_t)std::min<unsigned long long>((n16 + 1023) / 1024, 148ull * 16ull);
    if (gx == 0) gx = 1;
    dim3 grid(gx, B);
    if (fmt == PGG_FMT_U8)
        pgg::density_kernel<pgg::kFmtU8><<<grid, 256, 0, stream>>>(d_lats, lb, d_out, out_stride);
    else
        pgg::density_kernel<pgg::kFmtBits><<<grid, 256, 0, stream>>>(d_lats, lb, d_out, out_stride);
    PGG_LAUNCHED();
    return PGG_OK;
}

// The sweep proper for B lattices (B = 1: pgg_sweep).
// game = pgg::kGamePGG: h_r[b] = synergy factor of lattice b.  game = pgg::kGamePD (B = 1): h_r = {R, S, T, P}.
int32_t run_sweeps(uint8_t* d_lats, int32_t fmt, uint32_t B, uint32_t L, const double* h_r, double K,
                   const uint64_t* h_seeds, int32_t order_mode, double rho0, uint32_t t_begin,
                   uint32_t n_mcs, uint64_t* d_counts, cudaStream_t stream, int game = pgg::kGamePGG)
{
    const bool pd = game == pgg::kGamePD;
    if (pd && order_mode == PGG_ORDER_DTILE)
        return fail(PGG_ERR_UNSUPPORTED, "the prisoner's dilemma runs under the 16-sublattice schedule only");
    if (order_mode != PGG_ORDER_IID && order_mode != PGG_ORDER_PERM && order_mode != PGG_ORDER_DTILE)
        return fail(PGG_ERR_UNSUPPORTED, "unknown order_mode %d", order_mode);
    if (order_mode == PGG_ORDER_DTILE && L % 8 != 0)
        return fail(PGG_ERR_BAD_L, "L = %u: the double tiling schedule needs L %% 8 == 0 (PAPER.md:93)", L);
    if (!(K > 0.0) || !std::isfinite(K)) return fail(PGG_ERR_BAD_PARAM, "K must be finite and > 0");
    for (uint32_t b = 0; b < (pd ? 4u : B); ++b)
        if (!std::isfinite(h_r[b])) return fail(PGG_ERR_BAD_PARAM, pd ? "payoff %u (R, S, T, P) is not finite" : "r[%u] is not finite", b);
    if ((unsigned long long)t_begin + n_mcs > 4294967296ull)
        return fail(PGG_ERR_BAD_PARAM, "t_begin + n_mcs exceeds 2^32");

    int variant = order_mode == PGG_ORDER_DTILE ? PGG_VARIANT_DTILE : g_variant.load();
    const bool tile_ok = pgg::tile_supported(fmt, L);
    const bool band_ok = pgg::band_supported(fmt, L);
    const bool ring_ok = pgg::ring_supported(fmt, L);
    // measured (DESIGN.md appendix A): small lattices stay resident in shared memory;
    // of the streaming kernels uint8 is fastest on RING, bit-packed on BAND
    const bool res_ok = pgg::resident_supported(fmt, L);
    if (variant == PGG_VARIANT_AUTO) {
        // Measured rule (DESIGN.md appendix B, us per phase at r = 3.8).  RESIDENT takes one SM
        // per lattice whatever B is and grows with L^2 (1.5 us at L = 128, 2.8 at 320, 4.7 at 400, 6.9 at
        // 512); a V0 launch costs 4.2 us until B L^2 makes it throughput-bound.  So RESIDENT for L <= 320,
        // and above that from the batch size at which V0 has become slower: 3 lattices (L <= 448), 6 (L = 512).
        // uint8 L = 512 is also a whole-row strip for RING (4.2 us at B = 1, 6.8 at 13, 9.2 at 52): RING below
        // 20 lattices, RESIDENT from there (config 4).
        const bool ring_512 = fmt == PGG_FMT_U8 && L == 512 && ring_ok && B < 20;
        const bool res_pays = L <= 320 || (!ring_512 && B >= (L <= 448 ? 3u : 6u));
        // the streaming kernels need long rows (or whole-row strips: uint8 L = 512 * 2^k) to beat
        // V0's launch-bound 4-5 us; below that their fixed cost is ~9.5 us per launch
        const bool stream_pays = L >= 2048 || (fmt == PGG_FMT_U8 && L >= 512 && (L & (L - 1)) == 0);
        // bit-packed: LEAN (rows stream into a bit ring, queue lifetime of several steps) measured 2-3x
        // faster than BAND on ensembles and sparse states and level with it on the dense C5 lattice
        const bool lean_bits = fmt == PGG_FMT_BITS && pgg::lean_supported(fmt, L);
        // CLUSTER (the lattice resident in a CTA cluster's shared memory for the whole call; appendix B):
        // L = 512: 2.3-3.6 us per phase against RESIDENT's 5.3-6.9 and RING's 4.2-9.2 at every batch size;
        // L = 1024: 2.8 against 4.3 for one lattice, 8.7 against 11.9 for 64; L = 2048 from 32 lattices
        // (28.7 against 33 / 52 at 64); never at L = 4096 (16 CTAs per lattice leave the GPU idle)
        const bool cluster_pays = pgg::cluster_supported(fmt, L) && (L == 512 || L == 1024 || (L == 2048 && B >= 32));
        // uint8 at L >= 2048 (powers of two): a bit-packed working copy for the length of the call and LEAN on it
        // (PACKED).  The copy is 1/8 of the lattice -- 32 MiB at L = 16384, L2-resident -- and LEAN's phase on
        // it takes 45 us against RING's 60 on the uint8 rows; packing and unpacking cost two passes per CALL.
        static const uint32_t packed_min_L = [] { const char* e = getenv("PGG_PACKED_MIN_L"); return e ? (uint32_t)atoi(e) : 2048u; }();
        const bool packed_pays = fmt == PGG_FMT_U8 && !pd && pgg::lean_supported(PGG_FMT_BITS, L) && L >= packed_min_L;
        variant = cluster_pays ? PGG_VARIANT_CLUSTER
                : (res_ok && res_pays) ? PGG_VARIANT_RESIDENT
                : lean_bits ? PGG_VARIANT_LEAN
                : packed_pays ? PGG_VARIANT_PACKED
                : !stream_pays ? PGG_VARIANT_V0
                : (fmt == PGG_FMT_U8 && ring_ok) ? PGG_VARIANT_RING : band_ok ? PGG_VARIANT_BAND : PGG_VARIANT_V0;
    }
    if (pd) {  // two kernels carry the second game: LEAN where it runs, else the general V0
        const int asked = g_variant.load();
        if (asked != PGG_VARIANT_AUTO && asked != PGG_VARIANT_V0 && asked != PGG_VARIANT_LEAN && asked != PGG_VARIANT_PERSIST &&
            asked != PGG_VARIANT_CLUSTER)
            return fail(PGG_ERR_UNSUPPORTED, "the prisoner's dilemma runs on variants V0, LEAN, PERSIST and CLUSTER only (asked: %d)", asked);
        variant = asked == PGG_VARIANT_PERSIST ? PGG_VARIANT_PERSIST
                : asked == PGG_VARIANT_CLUSTER ? PGG_VARIANT_CLUSTER
                : (asked == PGG_VARIANT_AUTO && (L == 512 || L == 1024)) ? PGG_VARIANT_CLUSTER
                : (asked != PGG_VARIANT_V0 && pgg::lean_supported(fmt, L)) ? PGG_VARIANT_LEAN : PGG_VARIANT_V0;
        if (asked == PGG_VARIANT_LEAN && variant != PGG_VARIANT_LEAN)
            return fail(PGG_ERR_UNSUPPORTED, "variant %d does not support fmt %d, L %u", asked, fmt, L);
    }
    if (variant == PGG_VARIANT_RESIDENT && !res_ok)
        return fail(PGG_ERR_UNSUPPORTED, "variant %d does not support fmt %d, L %u", variant, fmt, L);
    if (variant == PGG_VARIANT_LEAN && !pgg::lean_supported(fmt, L))
        return fail(PGG_ERR_UNSUPPORTED, "variant %d does not support fmt %d, L %u", variant, fmt, L);
    if (variant == PGG_VARIANT_PACKED && !(fmt == PGG_FMT_U8 && !pd && pgg::lean_supported(PGG_FMT_BITS, L)))
        return fail(PGG_ERR_UNSUPPORTED, "variant %d does not support fmt %d, L %u", variant, fmt, L);
    if (variant == PGG_VARIANT_CLUSTER && !pgg::cluster_supported(fmt, L))
        return fail(PGG_ERR_UNSUPPORTED, "variant %d does not support fmt %d, L %u", variant, fmt, L);
    if (variant == PGG_VARIANT_PERSIST && !pgg::lean_persist_supported(fmt, L, B))
        return fail(PGG_ERR_UNSUPPORTED, "variant %d does not support fmt %d, L %u, B %u", variant, fmt, L, B);
    const bool split_ok = pgg::split_supported(fmt, L);
    if ((variant == PGG_VARIANT_BAND && !band_ok) || (variant == PGG_VARIANT_RING && !ring_ok) ||
        (variant == PGG_VARIANT_SPLIT && !split_ok) || (variant == PGG_VARIANT_DYN && !pgg::dyn_supported(fmt, L)))
        return fail(PGG_ERR_UNSUPPORTED, "variant %d does not support fmt %d, L %u", variant, fmt, L);
    if ((variant == PGG_VARIANT_TILE || variant == PGG_VARIANT_PIPE) && !tile_ok)
        return fail(PGG_ERR_UNSUPPORTED, "variant %d does not support fmt %d, L %u", variant, fmt, L);
    g_variant_used = variant;
    // PACKED: the kernels see a bit-packed working copy and run LEAN; the caller's layout stays uint8
    const bool packed = variant == PGG_VARIANT_PACKED;
    const int kfmt = packed ? PGG_FMT_BITS : fmt;
    if (packed) variant = PGG_VARIANT_LEAN;

    Scratch tmp(stream);
    // per-lattice seeds and acceptance tables
    std::vector<uint32_t> h_tables((size_t)B * pgg::kTableSize);
    for (uint32_t b = 0; b < B; ++b) {
        int32_t rc = pd ? pgg_pd_build_accept_table(h_r[0], h_r[1], h_r[2], h_r[3], K, h_tables.data() + (size_t)b * pgg::kTableSize)
                        : pgg_build_accept_table(h_r[b], K, h_tables.data() + (size_t)b * pgg::kTableSize);
        if (rc != PGG_OK) return rc;
    }
    uint64_t* d_seeds = nullptr;
    uint32_t* d_tables = nullptr;
    PGG_CUDA(tmp.alloc((void**)&d_seeds, sizeof(uint64_t) * B));
    PGG_CUDA(tmp.alloc((void**)&d_tables, sizeof(uint32_t) * h_tables.size()));
    {   // as kernel arguments: nothing is copied from pageable memory, the host vectors may die at scope exit
        int32_t rc = upload_params(B, h_seeds, h_tables.data(), d_seeds, d_tables, stream);
        if (rc != PGG_OK) return rc;
    }

    if (rho0 >= 0.0) {
        int32_t rc = launch_init(d_lats, fmt, B, L, rho0, d_seeds, stream);
        if (rc != PGG_OK) return rc;
    }
    if (n_mcs == 0) return PGG_OK;

    unsigned long long* d_count0 = nullptr;
    if (d_counts != nullptr) {
        PGG_CUDA(tmp.alloc((void**)&d_count0, sizeof(unsigned long long) * B));
        PGG_CUDA(cudaMemsetAsync(d_count0, 0, sizeof(unsigned long long) * B, stream));
        PGG_CUDA(cudaMemsetAsync(d_counts, 0, sizeof(uint64_t) * (size_t)B * n_mcs, stream));
        int32_t rc = launch_density(d_lats, fmt, B, L, d_count0, 1, stream);
        if (rc != PGG_OK) return rc;
    }

    const uint32_t chunk = std::min<uint32_t>(n_mcs, 4096u);
    if (variant == PGG_VARIANT_DTILE) {  // the paper's schedule: four parts per MCS, no class order
        pgg::PhaseArgs a{};
        a.lats = d_lats;
        a.lat_bytes = lattice_bytes(fmt, L);
        a.seeds = d_seeds;
        a.tables = d_tables;
        a.deltas = reinterpret_cast<unsigned long long*>(d_counts);
        a.L = L;
        a.n_mcs = n_mcs;
        a.t_begin = t_begin;
        for (uint32_t m = 0; m < n_mcs; ++m)
            for (uint32_t q = 0; q < 4; ++q) {
                pgg::dtile_launch(fmt, a, m, q, B, stream);
                PGG_LAUNCHED();
            }
        if (d_counts != nullptr) {
            pgg::finalize_counts_kernel<<<B, 1024, 0, stream>>>(
                reinterpret_cast<unsigned long long*>(d_counts), n_mcs, d_count0);
            PGG_LAUNCHED();
        }
        return PGG_OK;
    }
    uint8_t* d_order = nullptr;
    PGG_CUDA(tmp.alloc((void**)&d_order, (size_t)B * chunk * 16));
    uint8_t* d_work = d_lats;
    const unsigned long long n_words = (unsigned long long)B * L * L / 32ull;
    if (packed) {
        PGG_CUDA(tmp.alloc((void**)&d_work, (size_t)(4ull * n_words)));
        pgg::packed_launch(true, d_lats, d_work, n_words, stream);
        PGG_LAUNCHED();
    }

    pgg::PhaseArgs a;
    a.lats = d_work;
    a.lat_bytes = lattice_bytes(kfmt, L);
    a.seeds = d_seeds;
    a.tables = d_tables;
    a.order = d_order;
    a.deltas = reinterpret_cast<unsigned long long*>(d_counts);
    a.L = L;
    a.order_stride = chunk;
    a.n_mcs = n_mcs;
    a.t_begin = t_begin;

    pgg::TilePlan plan;
    pgg::BandPlan bplan;
    pgg::RingPlan rplan;
    if (variant == PGG_VARIANT_DYN) {
        int32_t rc = pgg::dyn_plan(L, B, &rplan);
        if (rc != 0) return fail(PGG_ERR_CUDA, "dyn kernel setup failed: %s", cudaGetErrorString((cudaError_t)rc));
    }
    if (variant == PGG_VARIANT_SPLIT) {
        int32_t rc = pgg::split_plan(L, B, &rplan);
        if (rc != 0) return fail(PGG_ERR_CUDA, "split kernel setup failed: %s", cudaGetErrorString((cudaError_t)rc));
    }
    if (variant == PGG_VARIANT_RING) {
        int32_t rc = pgg::ring_plan(fmt, L, B, &rplan);
        if (rc != 0) return fail(PGG_ERR_CUDA, "ring kernel setup failed: %s", cudaGetErrorString((cudaError_t)rc));
    }
    if (variant == PGG_VARIANT_BAND) {
        int32_t rc = pgg::band_plan(fmt, L, B, &bplan);
        if (rc != 0) return fail(PGG_ERR_CUDA, "band kernel setup failed: %s", cudaGetErrorString((cudaError_t)rc));
    }
    if (variant == PGG_VARIANT_PIPE) {
        int32_t rc = pgg::pipe_plan(fmt, L, B, &plan);
        if (rc != 0) return fail(PGG_ERR_CUDA, "pipe kernel setup failed: %s", cudaGetErrorString((cudaError_t)rc));
    }
    if (variant == PGG_VARIANT_TILE) {
        int32_t rc = pgg::tile_plan(fmt, L, B, &plan);
        if (rc != 0) return fail(PGG_ERR_CUDA, "tile kernel setup failed: %s", cudaGetErrorString((cudaError_t)rc));
    }

    pgg::LeanPlan lplan;
    pgg::ClusterPlan cplan;
    if (variant == PGG_VARIANT_CLUSTER) {
        int32_t rc = pgg::cluster_plan(fmt, L, B, &cplan);
        if (rc != 0) return fail(PGG_ERR_CUDA, "cluster kernel setup failed: %s", cudaGetErrorString((cudaError_t)rc));
    }
    unsigned int* d_gbar = nullptr;
    const size_t gbar_bytes = sizeof(unsigned int) * (size_t)B * 160;  // one flag per band: nb <= SMs / B, at least 1
    if (variant == PGG_VARIANT_PERSIST) {
        PGG_CUDA(tmp.alloc((void**)&d_gbar, gbar_bytes));
    }
    if (variant == PGG_VARIANT_LEAN || variant == PGG_VARIANT_PERSIST) {
        int32_t rc = pgg::lean_plan(kfmt, L, B, &lplan);
        if (rc != 0) return fail(PGG_ERR_CUDA, "lean kernel setup failed: %s", cudaGetErrorString((cudaError_t)rc));
    }
    pgg::ResPlan resplan;
    if (variant == PGG_VARIANT_RESIDENT) {
        int32_t rc = pgg::resident_plan(fmt, L, &resplan);
        if (rc != 0) return fail(PGG_ERR_CUDA, "resident kernel setup failed: %s", cudaGetErrorString((cudaError_t)rc));
    }
    for (uint32_t m0 = 0; m0 < n_mcs; m0 += chunk) {
        const uint32_t n_chunk = std::min<uint32_t>(chunk, n_mcs - m0);
        pgg::order_kernel<<<(B * n_chunk + 127) / 128, 128, 0, stream>>>(
            d_seeds, B, t_begin + m0, n_chunk, chunk, order_mode, d_order);
        PGG_LAUNCHED();
        if (variant == PGG_VARIANT_RESIDENT) {  // all 16 * n_chunk phases in one launch
            pgg::resident_launch(resplan, fmt, a, m0, n_chunk, B, stream);
            PGG_LAUNCHED();
            continue;
        }
        if (variant == PGG_VARIANT_CLUSTER) {   // likewise; the lattice stays in the cluster's shared memory
            PGG_CUDA(pgg::cluster_launch(cplan, fmt, a, m0, n_chunk, B, stream, game));
            PGG_LAUNCHED();
            continue;
        }
        if (variant == PGG_VARIANT_PERSIST) {   // likewise, cooperative: a barrier per phase instead of a launch
            PGG_CUDA(cudaMemsetAsync(d_gbar, 0, gbar_bytes, stream));
            PGG_CUDA(pgg::lean_persist_launch(lplan, a, m0, n_chunk, B, d_gbar, stream, game));
            PGG_LAUNCHED();
            continue;
        }
        for (uint32_t m = m0; m < m0 + n_chunk; ++m) {
            for (uint32_t k = 0; k < 16; ++k) {
                if (variant == PGG_VARIANT_LEAN) {
                    pgg::lean_launch(lplan, kfmt, a, m, k, B, stream, game);
                } else if (variant == PGG_VARIANT_DYN) {
                    pgg::dyn_launch(rplan, a, m, k, B, stream);
                } else if (variant == PGG_VARIANT_SPLIT) {
                    pgg::split_launch(rplan, a, m, k, B, stream);
                } else if (variant == PGG_VARIANT_RING) {
                    pgg::ring_launch(rplan, fmt, a, m, k, B, stream);
                } else if (variant == PGG_VARIANT_BAND) {
                    pgg::band_launch(bplan, fmt, a, m, k, B, stream);
                } else if (variant == PGG_VARIANT_PIPE) {
                    pgg::pipe_launch(plan, fmt, a, m, k, B, stream);
                } else if (variant == PGG_VARIANT_TILE) {
                    pgg::tile_launch(plan, fmt, a, m, k, B, stream);
                } else {
                    const uint32_t n_cls = (L / 4) * (L / 4);
                    dim3 grid((n_cls + 255) / 256, B);
                    if (pd && fmt == PGG_FMT_U8)
                        pgg::phase_v0_kernel<pgg::kFmtU8, pgg::kGamePD><<<grid, 256, 0, stream>>>(a, m, k);
                    else if (pd)
                        pgg::phase_v0_kernel<pgg::kFmtBits, pgg::kGamePD><<<grid, 256, 0, stream>>>(a, m, k);
                    else if (fmt == PGG_FMT_U8)
                        pgg::phase_v0_kernel<pgg::kFmtU8><<<grid, 256, 0, stream>>>(a, m, k);
                    else
                        pgg::phase_v0_kernel<pgg::kFmtBits><<<grid, 256, 0, stream>>>(a, m, k);
                }
                PGG_LAUNCHED();
            }
        }
    }
    if (packed) {  // the working copy -> the caller's uint8 lattice
        pgg::packed_launch(false, d_lats, d_work, n_words, stream);
        PGG_LAUNCHED();
    }
    if (d_counts != nullptr) {
        pgg::finalize_counts_kernel<<<B, 1024, 0, stream>>>(
            reinterpret_cast<unsigned long long*>(d_counts), n_mcs, d_count0);
        PGG_LAUNCHED();
    }
    return PGG_OK;
}

// ---- pgg_sweep_static: the temporaries of a one-lattice sweep in a file-scope device array --------
// Layout (bytes): [0, 8) seed | [8, 16) initial cooperator count | [256, 868) acceptance table |
// [1024, 1024 + 16 * PGG_STATIC_MAX_MCS) phase-class order.  In HOST code the name below is a host-side
// stand-in, not a device address: only the pointer cudaGetSymbolAddress returns may go to a kernel.
constexpr size_t kStaticSeedOff = 0, kStaticCount0Off = 8, kStaticTableOff = 256, kStaticOrderOff = 1024;
static_assert(kStaticTableOff + sizeof(uint32_t) * pgg::kTableSize <= kStaticOrderOff, "table overlaps the order");
static __device__ __align__(256) unsigned char g_static_scratch[PGG_STATIC_SCRATCH_BYTES];

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
unsigned char* g_static_ptr[kStaticMaxDevices] = {};  // per device, resolved once with that device current

// Device address of g_static_scratch on the CURRENT device (no allocation: the array is part of the module).
int32_t static_scratch(unsigned char** out)
{
    int dev = -1;
    PGG_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(PGG_ERR_UNSUPPORTED, "device ordinal %d: at most %d devices", dev, kStaticMaxDevices);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (g_static_ptr[dev] == nullptr) {
        void* p = nullptr;
        PGG_CUDA(cudaGetSymbolAddress(&p, g_static_scratch));
        if (p == nullptr || (reinterpret_cast<uintptr_t>(p) & 255u) != 0)
            return fail(PGG_ERR_CUDA, "cudaGetSymbolAddress returned %p for the static scratch", p);
        g_static_ptr[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_static_ptr[dev];
    return PGG_OK;
}

}  // namespace

extern "C" {

int32_t pgg_sweep_static(void* d_lat, int32_t fmt, uint32_t L, double r, double K, uint64_t seed,
                         int32_t order_mode, uint32_t t_begin, uint32_t n_mcs, uint64_t* d_counts, void* stream_)
{
    int32_t rc = check_lattice_args(d_lat, fmt, L);
    if (rc != PGG_OK) return rc;
    if (order_mode == PGG_ORDER_DTILE)
        return fail(PGG_ERR_UNSUPPORTED, "pgg_sweep_static runs the 16-sublattice schedule only (PGG_ORDER_IID / PGG_ORDER_PERM)");
    if (order_mode != PGG_ORDER_IID && order_mode != PGG_ORDER_PERM)
        return fail(PGG_ERR_UNSUPPORTED, "unknown order_mode %d", order_mode);
    if (!(K > 0.0) || !std::isfinite(K)) return fail(PGG_ERR_BAD_PARAM, "K must be finite and > 0");
    if (!std::isfinite(r)) return fail(PGG_ERR_BAD_PARAM, "r is not finite");
    if ((unsigned long long)t_begin + n_mcs > 4294967296ull)
        return fail(PGG_ERR_BAD_PARAM, "t_begin + n_mcs exceeds 2^32");
    if (n_mcs > PGG_STATIC_MAX_MCS)
        return fail(PGG_ERR_BAD_PARAM, "n_mcs = %u exceeds PGG_STATIC_MAX_MCS = %u: the static scratch holds the class order "
                    "of %u MCS; split the run into several calls", n_mcs, PGG_STATIC_MAX_MCS, PGG_STATIC_MAX_MCS);
    if (n_mcs == 0) return PGG_OK;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);

    // the kernel pgg_sweep's AUTO rule picks for ONE lattice (run_sweeps above), among the five this entry point carries
    int variant = g_variant.load();
    if (variant == PGG_VARIANT_AUTO) {
        const bool stream_pays = L >= 2048 || (fmt == PGG_FMT_U8 && L >= 512 && (L & (L - 1)) == 0);
        variant = (pgg::cluster_supported(fmt, L) && (L == 512 || L == 1024)) ? PGG_VARIANT_CLUSTER
                : (pgg::resident_supported(fmt, L) && L <= 320) ? PGG_VARIANT_RESIDENT
                : (fmt == PGG_FMT_BITS && pgg::lean_supported(fmt, L)) ? PGG_VARIANT_LEAN
                : (stream_pays && fmt == PGG_FMT_U8 && pgg::ring_supported(fmt, L)) ? PGG_VARIANT_RING : PGG_VARIANT_V0;
    }
    const bool ok = variant == PGG_VARIANT_V0 || (variant == PGG_VARIANT_CLUSTER && pgg::cluster_supported(fmt, L)) ||
                    (variant == PGG_VARIANT_RESIDENT && pgg::resident_supported(fmt, L)) ||
                    (variant == PGG_VARIANT_LEAN && pgg::lean_supported(fmt, L)) ||
                    (variant == PGG_VARIANT_RING && pgg::ring_supported(fmt, L));
    if (!ok) return fail(PGG_ERR_UNSUPPORTED, "pgg_sweep_static: variant %d is not available for fmt %d, L %u", variant, fmt, L);
    g_variant_used = variant;

    unsigned char* scratch = nullptr;
    rc = static_scratch(&scratch);
    if (rc != PGG_OK) return rc;
    uint64_t* d_seed = reinterpret_cast<uint64_t*>(scratch + kStaticSeedOff);
    unsigned long long* d_count0 = reinterpret_cast<unsigned long long*>(scratch + kStaticCount0Off);
    uint32_t* d_table = reinterpret_cast<uint32_t*>(scratch + kStaticTableOff);
    uint8_t* d_order = scratch + kStaticOrderOff;

    uint32_t h_table[pgg::kTableSize];
    rc = pgg_build_accept_table(r, K, h_table);
    if (rc != PGG_OK) return rc;
    rc = upload_params(1, &seed, h_table, d_seed, d_table, stream);  // kernel arguments: no staging buffer
    if (rc != PGG_OK) return rc;

    uint8_t* d_lats = static_cast<uint8_t*>(d_lat);
    if (d_counts != nullptr) {
        PGG_CUDA(cudaMemsetAsync(d_count0, 0, sizeof(unsigned long long), stream));  // the array keeps the last call's value
        PGG_CUDA(cudaMemsetAsync(d_counts, 0, sizeof(uint64_t) * (size_t)n_mcs, stream));
        rc = launch_density(d_lats, fmt, 1, L, d_count0, 1, stream);
        if (rc != PGG_OK) return rc;
    }

    pgg::PhaseArgs a;
    a.lats = d_lats;
    a.lat_bytes = lattice_bytes(fmt, L);
    a.seeds = d_seed;
    a.tables = d_table;
    a.order = d_order;
    a.deltas = reinterpret_cast<unsigned long long*>(d_counts);
    a.L = L;
    a.order_stride = n_mcs;
    a.n_mcs = n_mcs;
    a.t_begin = t_begin;

    pgg::order_kernel<<<(n_mcs + 127) / 128, 128, 0, stream>>>(d_seed, 1, t_begin, n_mcs, n_mcs, order_mode, d_order);
    PGG_LAUNCHED();
    if (variant == PGG_VARIANT_RESIDENT) {
        pgg::ResPlan plan;
        int32_t e = pgg::resident_plan(fmt, L, &plan);
        if (e != 0) return fail(PGG_ERR_CUDA, "resident kernel setup failed: %s", cudaGetErrorString((cudaError_t)e));
        pgg::resident_launch(plan, fmt, a, 0, n_mcs, 1, stream);
        PGG_LAUNCHED();
    } else if (variant == PGG_VARIANT_CLUSTER) {
        pgg::ClusterPlan plan;
        int32_t e = pgg::cluster_plan(fmt, L, 1, &plan);
        if (e != 0) return fail(PGG_ERR_CUDA, "cluster kernel setup failed: %s", cudaGetErrorString((cudaError_t)e));
        PGG_CUDA(pgg::cluster_launch(plan, fmt, a, 0, n_mcs, 1, stream, pgg::kGamePGG));
        PGG_LAUNCHED();
    } else {
        pgg::LeanPlan lplan;
        pgg::RingPlan rplan;
        if (variant == PGG_VARIANT_LEAN) {
            int32_t e = pgg::lean_plan(fmt, L, 1, &lplan);
            if (e != 0) return fail(PGG_ERR_CUDA, "lean kernel setup failed: %s", cudaGetErrorString((cudaError_t)e));
        }
        if (variant == PGG_VARIANT_RING) {
            int32_t e = pgg::ring_plan(fmt, L, 1, &rplan);
            if (e != 0) return fail(PGG_ERR_CUDA, "ring kernel setup failed: %s", cudaGetErrorString((cudaError_t)e));
        }
        for (uint32_t m = 0; m < n_mcs; ++m)
            for (uint32_t k = 0; k < 16; ++k) {
                if (variant == PGG_VARIANT_LEAN) {
                    pgg::lean_launch(lplan, fmt, a, m, k, 1, stream, pgg::kGamePGG);
                } else if (variant == PGG_VARIANT_RING) {
                    pgg::ring_launch(rplan, fmt, a, m, k, 1, stream);
                } else {
                    const uint32_t n_cls = (L / 4) * (L / 4);
                    dim3 grid((n_cls + 255) / 256, 1);
                    if (fmt == PGG_FMT_U8)
                        pgg::phase_v0_kernel<pgg::kFmtU8><<<grid, 256, 0, stream>>>(a, m, k);
                    else
                        pgg::phase_v0_kernel<pgg::kFmtBits><<<grid, 256, 0, stream>>>(a, m, k);
                }
                PGG_LAUNCHED();
            }
    }
    if (d_counts != nullptr) {
        pgg::finalize_counts_kernel<<<1, 1024, 0, stream>>>(reinterpret_cast<unsigned long long*>(d_counts), n_mcs, d_count0);
        PGG_LAUNCHED();
    }
    return PGG_OK;
}

int32_t pgg_build_accept_table(double r, double K, uint32_t* h_out153)
{
    if (h_out153 == nullptr) return fail(PGG_ERR_NULL, "out153 is NULL");
    if (!std::isfinite(r) || !std::isfinite(K) || !(K > 0.0))
        return fail(PGG_ERR_BAD_PARAM, "r and K must be finite, K > 0");
    // Eq. (3), in the operation order of SURVEY 8(c) D3.  Pi_x - Pi_y =
    // (r/5)(A_x - A_y) - 5 (s_x - s_y) because Pi = (r/5) A - 5 s (c = 1).
    for (int ds = -1; ds <= 1; ++ds) {
        for (int dA = -25; dA <= 25; ++dA) {
            volatile double delta = (r * (double)dA) / 5.0 - 5.0 * (double)ds;
            volatile double z = delta / K;
            volatile double W = 1.0 / (1.0 + std::exp(z));
            const double v = W * 4294967296.0;
            h_out153[(ds + 1) * 51 + (dA + 25)] =
                (v >= 4294967295.0) ? 0xFFFFFFFFu : (uint32_t)std::floor(v);
        }
    }
    return PGG_OK;
}

int32_t pgg_pd_build_accept_table(double R, double S, double T, double P, double K, uint32_t* h_out50)
{
    if (h_out50 == nullptr) return fail(PGG_ERR_NULL, "out50 is NULL");
    if (!std::isfinite(R) || !std::isfinite(S) || !std::isfinite(T) || !std::isfinite(P) || !std::isfinite(K) || !(K > 0.0))
        return fail(PGG_ERR_BAD_PARAM, "R, S, T, P and K must be finite, K > 0");
    // Eq. (3), for the pair-game payoffs of PAPER.md:131 (readings G1, G3 in pgg.h)
    for (int sx = 0; sx <= 1; ++sx)
        for (int nx = 0; nx <= 4; ++nx)
            for (int ny = 0; ny <= 4; ++ny) {
                auto pay = [&](int s, int n) { return s == 1 ? R * (double)n + S * (double)(4 - n) : T * (double)n + P * (double)(4 - n); };
                volatile double px = pay(sx, nx);
                volatile double py = pay(1 - sx, ny);
                volatile double z = (px - py) / K;
                volatile double W = 1.0 / (1.0 + std::exp(z));
                const double v = W * 4294967296.0;
                h_out50[sx * 25 + nx * 5 + ny] = (v >= 4294967295.0) ? 0xFFFFFFFFu : (uint32_t)std::floor(v);
            }
    return PGG_OK;
}

int32_t pgg_pd_sweep(void* d_lat, int32_t fmt, uint32_t L, double R, double S, double T, double P, double K,
                     uint64_t seed, int32_t order_mode, uint32_t t_begin, uint32_t n_mcs, uint64_t* d_counts,
                     void* stream)
{
    int32_t rc = check_lattice_args(d_lat, fmt, L);
    if (rc != PGG_OK) return rc;
    const double h_pd[4] = {R, S, T, P};
    return run_sweeps(static_cast<uint8_t*>(d_lat), fmt, 1, L, h_pd, K, &seed, order_mode, -1.0, t_begin, n_mcs,
                      d_counts, static_cast<cudaStream_t>(stream), pgg::kGamePD);
}

int32_t pgg_init_lattice(void* d_lat, int32_t fmt, uint32_t L, double rho0, uint64_t seed, void* stream)
{
    int32_t rc = check_lattice_args(d_lat, fmt, L);
    if (rc != PGG_OK) return rc;
    if (!(rho0 >= 0.0 && rho0 <= 1.0)) return fail(PGG_ERR_BAD_PARAM, "rho0 must lie in [0,1]");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    Scratch tmp(s);
    uint64_t* d_seed = nullptr;
    PGG_CUDA(tmp.alloc((void**)&d_seed, sizeof(uint64_t)));
    rc = upload_params(1, &seed, nullptr, d_seed, nullptr, s);
    if (rc != PGG_OK) return rc;
    return launch_init(static_cast<uint8_t*>(d_lat), fmt, 1, L, rho0, d_seed, s);
}

int32_t pgg_sweep(void* d_lat, int32_t fmt, uint32_t L, double r, double K, uint64_t seed,
                  int32_t order_mode, uint32_t t_begin, uint32_t n_mcs, uint64_t* d_counts, void* stream)
{
    int32_t rc = check_lattice_args(d_lat, fmt, L);
    if (rc != PGG_OK) return rc;
    return run_sweeps(static_cast<uint8_t*>(d_lat), fmt, 1, L, &r, K, &seed, order_mode, -1.0, t_begin,
                      n_mcs, d_counts, static_cast<cudaStream_t>(stream));
}

int32_t pgg_density(const void* d_lat, int32_t fmt, uint32_t L, uint64_t* d_count, void* stream)
{
    int32_t rc = check_lattice_args(d_lat, fmt, L);
    if (rc != PGG_OK) return rc;
    if (d_count == nullptr) return fail(PGG_ERR_NULL, "d_count is NULL");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    PGG_CUDA(cudaMemsetAsync(d_count, 0, sizeof(uint64_t), s));
    return launch_density(static_cast<const uint8_t*>(d_lat), fmt, 1, L,
                          reinterpret_cast<unsigned long long*>(d_count), 1, s);
}

int32_t pgg_run_ensemble(void* d_lats, int32_t fmt, uint32_t B, uint32_t L, const double* h_r, double K,
                         const uint64_t* h_seeds, int32_t order_mode, double rho0, uint32_t t_begin,
                         uint32_t n_mcs, uint64_t* d_counts, void* stream)
{
    int32_t rc = check_lattice_args(d_lats, fmt, L);
    if (rc != PGG_OK) return rc;
    if (h_r == nullptr || h_seeds == nullptr) return fail(PGG_ERR_NULL, "h_r / h_seeds is NULL");
    if (B == 0 || B > 65535) return fail(PGG_ERR_BAD_PARAM, "B = %u: need 1 <= B <= 65535", B);
    if (rho0 > 1.0 || rho0 != rho0) return fail(PGG_ERR_BAD_PARAM, "rho0 must be <= 1 (or < 0 to continue)");
    return run_sweeps(static_cast<uint8_t*>(d_lats), fmt, B, L, h_r, K, h_seeds, order_mode, rho0,
                      t_begin, n_mcs, d_counts, static_cast<cudaStream_t>(stream));
}

int32_t pgg_phase_classes(uint64_t seed, uint32_t t, int32_t order_mode, uint8_t* h_out16, void* stream)
{
    if (h_out16 == nullptr) return fail(PGG_ERR_NULL, "h_out16 is NULL");
    if (order_mode != PGG_ORDER_IID && order_mode != PGG_ORDER_PERM)
        return fail(PGG_ERR_UNSUPPORTED, "unknown order_mode %d", order_mode);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    Scratch tmp(s);
    uint64_t* d_seed = nullptr;
    uint8_t* d_order = nullptr;
    PGG_CUDA(tmp.alloc((void**)&d_seed, sizeof(uint64_t)));
    PGG_CUDA(tmp.alloc((void**)&d_order, 16));
    {
        int32_t rc = upload_params(1, &seed, nullptr, d_seed, nullptr, s);
        if (rc != PGG_OK) return rc;
    }
    pgg::order_kernel<<<1, 128, 0, s>>>(d_seed, 1, t, 1, 1, order_mode, d_order);
    PGG_LAUNCHED();
    PGG_CUDA(cudaMemcpyAsync(h_out16, d_order, 16, cudaMemcpyDeviceToHost, s));
    PGG_CUDA(cudaStreamSynchronize(s));
    return PGG_OK;
}

int32_t pgg_set_variant(int32_t variant)
{
    if (variant < PGG_VARIANT_AUTO || variant > PGG_VARIANT_PACKED || variant == PGG_VARIANT_DTILE || variant == 3)
        return fail(PGG_ERR_UNSUPPORTED, "unknown variant %d", variant);
    g_variant.store(variant);
    return PGG_OK;
}

int32_t pgg_get_variant_used(void) { return g_variant_used; }

int32_t pgg_variant_supported(int32_t variant, int32_t fmt, uint32_t L)
{
    if (fmt != PGG_FMT_U8 && fmt != PGG_FMT_BITS) return 0;
    if (L < 4 || L % 4 != 0 || L >= 65536 || (fmt == PGG_FMT_BITS && L % 32 != 0)) return 0;
    if (variant == PGG_VARIANT_AUTO || variant == PGG_VARIANT_V0) return 1;
    if (variant == PGG_VARIANT_TILE || variant == PGG_VARIANT_PIPE) return pgg::tile_supported(fmt, L) ? 1 : 0;
    if (variant == PGG_VARIANT_BAND) return pgg::band_supported(fmt, L) ? 1 : 0;
    if (variant == PGG_VARIANT_RING) return pgg::ring_supported(fmt, L) ? 1 : 0;
    if (variant == PGG_VARIANT_SPLIT) return pgg::split_supported(fmt, L) ? 1 : 0;
    if (variant == PGG_VARIANT_DYN) return pgg::dyn_supported(fmt, L) ? 1 : 0;
    if (variant == PGG_VARIANT_RESIDENT) return pgg::resident_supported(fmt, L) ? 1 : 0;
    if (variant == PGG_VARIANT_LEAN) return pgg::lean_supported(fmt, L) ? 1 : 0;
    if (variant == PGG_VARIANT_PERSIST) return pgg::lean_persist_supported(fmt, L, 1) ? 1 : 0;
    if (variant == PGG_VARIANT_CLUSTER) return pgg::cluster_supported(fmt, L) ? 1 : 0;
    if (variant == PGG_VARIANT_PACKED) return (fmt == PGG_FMT_U8 && pgg::lean_supported(PGG_FMT_BITS, L)) ? 1 : 0;
    return 0;
}

int32_t pgg_probe_draw_rate(uint32_t iters, uint64_t seed, uint64_t* h_n_draws, void* stream)
{
    if (h_n_draws == nullptr) return fail(PGG_ERR_NULL, "h_n_draws is NULL");
    if (iters == 0) return fail(PGG_ERR_BAD_PARAM, "iters must be > 0");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int dev = 0, sms = 0;
    PGG_CUDA(cudaGetDevice(&dev));
    PGG_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const uint32_t grid = (uint32_t)sms * 4u;  // 4 CTAs of 256 threads per SM: every SM full at 64 registers
    Scratch tmp(s);
    uint32_t* d_sink = nullptr;
    PGG_CUDA(tmp.alloc((void**)&d_sink, sizeof(uint32_t) * grid * pgg::kProbeThreads));
    const pgg::StepKey sk = pgg::make_step_key(seed, 0u, 0u, 0u);
    pgg::draw_ceiling_kernel<<<grid, pgg::kProbeThreads, 0, s>>>(sk, iters, d_sink);
    PGG_LAUNCHED();
    *h_n_draws = 2ull * iters * grid * pgg::kProbeThreads;
    return PGG_OK;
}

int32_t pgg_count_interface(const void* d_lat, int32_t fmt, uint32_t L, uint64_t* d_count, void* stream)
{
    int32_t rc = check_lattice_args(d_lat, fmt, L);
    if (rc != PGG_OK) return rc;
    if (d_count == nullptr) return fail(PGG_ERR_NULL, "d_count is NULL");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    PGG_CUDA(cudaMemsetAsync(d_count, 0, sizeof(uint64_t), s));
    const uint32_t n = L * L;
    const uint32_t grid = std::min<uint32_t>((n + 255u) / 256u, 148u * 32u);
    if (fmt == PGG_FMT_U8)
        pgg::interface_count_kernel<pgg::kFmtU8><<<grid, 256, 0, s>>>(static_cast<const uint8_t*>(d_lat), L,
                                                                    reinterpret_cast<unsigned long long*>(d_count));
    else
        pgg::interface_count_kernel<pgg::kFmtBits><<<grid, 256, 0, s>>>(static_cast<const uint8_t*>(d_lat), L,
                                                                      reinterpret_cast<unsigned long long*>(d_count));
    PGG_LAUNCHED();
    return PGG_OK;
}

// ---- row slabs of one lattice over several GPUs (kernels in pgg_kernels_slab.cuh) ----

uint64_t pgg_slab_bytes(int32_t fmt, uint32_t L, uint32_t n_rows)
{
    const unsigned long long row = fmt == PGG_FMT_U8 ? L : L / 8;
    return row * ((unsigned long long)n_rows + 6ull);
}

uint32_t pgg_slab_step_rows(int32_t fmt, uint32_t L)
{
    pgg::LeanPlan p{};
    if ((fmt != PGG_FMT_BITS && fmt != PGG_FMT_U8) || !pgg::lean_supported(fmt, L) || pgg::lean_plan(fmt, L, 1, &p) != 0) return 4;
    return 4 * p.R;
}

// game = pgg::kGamePGG: pay[0] = r.  game = pgg::kGamePD: pay = {R, S, T, P}.
static int32_t run_slab_sweep(void* d_slab, int32_t fmt, uint32_t L, uint32_t row0, uint32_t n_rows, int game, const double* pay,
                              double K, uint64_t seed, int32_t order_mode, uint32_t t_begin, uint32_t k_begin, uint32_t n_phases,
                              void* d_up_halo, void* d_dn_halo, uint32_t* d_flags, uint32_t* d_up_flag, uint32_t* d_dn_flag,
                              uint32_t epoch0, uint64_t* d_deltas, void* stream_)
{
    const bool pd = game == pgg::kGamePD;
    const double r = pay[0];
    int32_t rc = check_lattice_args(d_slab, fmt, L);
    if (rc != PGG_OK) return rc;
    if (d_up_halo == nullptr || d_dn_halo == nullptr) return fail(PGG_ERR_NULL, "halo pointer is NULL");
    const uintptr_t align = fmt == PGG_FMT_BITS ? 3u : 0u;  // bit rows are updated by 32-bit atomics
    if ((reinterpret_cast<uintptr_t>(d_up_halo) & align) || (reinterpret_cast<uintptr_t>(d_dn_halo) & align))
        return fail(PGG_ERR_ALIGN, "bit-packed halo rows must be 4-byte aligned");
    if (n_rows < 4 || n_rows % 4 != 0 || row0 % 4 != 0 || (unsigned long long)row0 + n_rows > L)
        return fail(PGG_ERR_BAD_PARAM, "slab rows [%u, %u + %u): need row0 %% 4 == 0, n_rows %% 4 == 0, n_rows >= 4, row0 + n_rows <= L = %u",
                    row0, row0, n_rows, L);
    if (order_mode != PGG_ORDER_IID && order_mode != PGG_ORDER_PERM)
        return fail(PGG_ERR_UNSUPPORTED, "slabs run the 16-sublattice schedule only (PGG_ORDER_IID / PGG_ORDER_PERM), not order_mode %d", order_mode);
    if (!(K > 0.0) || !std::isfinite(K)) return fail(PGG_ERR_BAD_PARAM, "K must be finite and > 0");
    for (int q = 0; q < (pd ? 4 : 1); ++q)
        if (!std::isfinite(pay[q])) return fail(PGG_ERR_BAD_PARAM, pd ? "a payoff (R, S, T, P) is not finite" : "r is not finite");
    if (k_begin >= 16) return fail(PGG_ERR_BAD_PARAM, "k_begin = %u: a MCS has phases 0 .. 15", k_begin);
    if (d_flags != nullptr && (d_up_flag == nullptr || d_dn_flag == nullptr))
        return fail(PGG_ERR_NULL, "d_flags given without both neighbour flag pointers");
    if (n_phases == 0) return PGG_OK;
    const unsigned long long n_span = ((unsigned long long)k_begin + n_phases + 15ull) / 16ull;  // MCS touched
    if (n_span > PGG_SLAB_MAX_MCS)
        return fail(PGG_ERR_BAD_PARAM, "the call spans %llu MCS, more than PGG_SLAB_MAX_MCS = %u: split it", n_span, PGG_SLAB_MAX_MCS);
    if ((unsigned long long)t_begin + n_span > 4294967296ull) return fail(PGG_ERR_BAD_PARAM, "t_begin + MCS spanned exceeds 2^32");
    if ((unsigned long long)epoch0 + n_phases > 4294967295ull) return fail(PGG_ERR_BAD_PARAM, "epoch0 + n_phases exceeds 2^32 - 1");
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);

    uint32_t h_table[pgg::kTableSize] = {};
    rc = pd ? pgg_pd_build_accept_table(pay[0], pay[1], pay[2], pay[3], K, h_table) : pgg_build_accept_table(r, K, h_table);
    if (rc != PGG_OK) return rc;
    Scratch tmp(stream);
    uint64_t* d_seed = nullptr;
    uint32_t* d_table = nullptr;
    uint8_t* d_order = nullptr;
    PGG_CUDA(tmp.alloc((void**)&d_seed, sizeof(uint64_t)));
    PGG_CUDA(tmp.alloc((void**)&d_table, sizeof(h_table)));
    PGG_CUDA(tmp.alloc((void**)&d_order, 16 * (size_t)n_span));
    rc = upload_params(1, &seed, h_table, d_seed, d_table, stream);
    if (rc != PGG_OK) return rc;
    pgg::order_kernel<<<((uint32_t)n_span + 127) / 128, 128, 0, stream>>>(d_seed, 1, t_begin, (uint32_t)n_span, (uint32_t)n_span,
                                                                         order_mode == PGG_ORDER_PERM ? 1 : 0, d_order);
    PGG_LAUNCHED();

    pgg::SlabArgs a{};
    a.slab = static_cast<uint8_t*>(d_slab);
    a.up_halo = static_cast<uint8_t*>(d_up_halo);
    a.dn_halo = static_cast<uint8_t*>(d_dn_halo);
    a.seed = d_seed;
    a.table = d_table;
    a.order = d_order;
    a.deltas = reinterpret_cast<unsigned long long*>(d_deltas);
    a.flags = d_flags;
    a.up_flag = d_up_flag;
    a.dn_flag = d_dn_flag;
    a.L = L;
    a.row0 = row0;
    a.n_rows = n_rows;
    a.t0 = t_begin;
    // Slabs of whole LEAN steps (L = 1024 .. 32768, a power of two): LEAN's ring kernel on the slab's buffer.
    static const bool slab_lean = [] { const char* e = getenv("PGG_SLAB_LEAN"); return e == nullptr || atoi(e) != 0; }();
    pgg::LeanPlan lplan{};
    const bool lean = slab_lean && pgg::lean_plan_slab(fmt, L, row0, n_rows, &lplan) == 0;
    g_variant_used = lean ? PGG_VARIANT_LEAN : PGG_VARIANT_V0;  // pgg_get_variant_used(): which slab kernel ran
    pgg::PhaseArgs pa{};
    if (lean) {
        // the address lattice row 0 would have: buffer row q holds lattice row row0 - 3 + q (rows never wrap in a slab)
        pa.lats = reinterpret_cast<uint8_t*>(reinterpret_cast<uintptr_t>(d_slab) - ((intptr_t)row0 - 3) * (intptr_t)(fmt == PGG_FMT_U8 ? L : L / 8));
        pa.lat_bytes = 0;
        pa.seeds = d_seed;
        pa.tables = d_table;
        pa.order = d_order;
        pa.deltas = reinterpret_cast<unsigned long long*>(d_deltas);
        pa.L = L;
        pa.order_stride = (uint32_t)n_span;
        pa.n_mcs = (uint32_t)n_span;
        pa.t_begin = t_begin;
    }
    // General kernels.  uint8: a thread per active site; bit-packed: a thread per 32-site word of an active row.  8 CTAs
    // of 256 threads per SM at most, grid-stride: the flag protocol costs one wait and one post per CTA.
    const uint32_t n_items = fmt == PGG_FMT_U8 ? (n_rows / 4) * (L / 4) : (n_rows / 4) * (L / 32);
    const dim3 grid(std::min<uint32_t>((n_items + 255) / 256, 148u * 8u));
    for (uint32_t p = 0; p < n_phases; ++p) {
        const uint32_t q = k_begin + p, t = t_begin + (q >> 4), k = q & 15u;
        if (lean)
            pgg::lean_slab_launch(lplan, fmt, pa, t - t_begin, k, a, epoch0 + p, stream, game);
        else if (fmt == PGG_FMT_U8 && pd)
            pgg::phase_slab_kernel<pgg::kFmtU8, pgg::kGamePD><<<grid, 256, 0, stream>>>(a, t, k, epoch0 + p);
        else if (fmt == PGG_FMT_U8)
            pgg::phase_slab_kernel<pgg::kFmtU8><<<grid, 256, 0, stream>>>(a, t, k, epoch0 + p);
        else if (pd)
            pgg::phase_slab_words_kernel<pgg::kGamePD><<<grid, 256, 0, stream>>>(a, t, k, epoch0 + p);
        else
            pgg::phase_slab_words_kernel<pgg::kGamePGG><<<grid, 256, 0, stream>>>(a, t, k, epoch0 + p);
        PGG_LAUNCHED();
    }
    return PGG_OK;
}

int32_t pgg_slab_sweep(void* d_slab, int32_t fmt, uint32_t L, uint32_t row0, uint32_t n_rows, double r, double K,
                       uint64_t seed, int32_t order_mode, uint32_t t_begin, uint32_t k_begin, uint32_t n_phases,
                       void* d_up_halo, void* d_dn_halo, uint32_t* d_flags, uint32_t* d_up_flag, uint32_t* d_dn_flag,
                       uint32_t epoch0, uint64_t* d_deltas, void* stream)
{
    return run_slab_sweep(d_slab, fmt, L, row0, n_rows, pgg::kGamePGG, &r, K, seed, order_mode, t_begin, k_begin, n_phases,
                          d_up_halo, d_dn_halo, d_flags, d_up_flag, d_dn_flag, epoch0, d_deltas, stream);
}

int32_t pgg_pd_slab_sweep(void* d_slab, int32_t fmt, uint32_t L, uint32_t row0, uint32_t n_rows, double R, double S, double T,
                          double P, double K, uint64_t seed, int32_t order_mode, uint32_t t_begin, uint32_t k_begin,
                          uint32_t n_phases, void* d_up_halo, void* d_dn_halo, uint32_t* d_flags, uint32_t* d_up_flag,
                          uint32_t* d_dn_flag, uint32_t epoch0, uint64_t* d_deltas, void* stream)
{
    const double pay[4] = {R, S, T, P};
    return run_slab_sweep(d_slab, fmt, L, row0, n_rows, pgg::kGamePD, pay, K, seed, order_mode, t_begin, k_begin, n_phases,
                          d_up_halo, d_dn_halo, d_flags, d_up_flag, d_dn_flag, epoch0, d_deltas, stream);
}

int32_t pgg_slab_alloc(uint64_t bytes, void** d_out)
{
    if (d_out == nullptr) return fail(PGG_ERR_NULL, "d_out is NULL");
    if (bytes == 0) return fail(PGG_ERR_BAD_PARAM, "bytes is 0");
    void* p = nullptr;
    PGG_CUDA(cudaMalloc(&p, bytes));
    cudaError_t e = cudaMemset(p, 0, bytes);
    if (e != cudaSuccess) {
        cudaFree(p);
        return fail(PGG_ERR_CUDA, "cudaMemset failed: %s", cudaGetErrorString(e));
    }
    *d_out = p;
    return PGG_OK;
}

int32_t pgg_slab_free(void* d_ptr)
{
    if (d_ptr != nullptr) PGG_CUDA(cudaFree(d_ptr));
    return PGG_OK;
}

int32_t pgg_slab_ipc_export(void* d_ptr, uint8_t* h_handle64)
{
    if (d_ptr == nullptr || h_handle64 == nullptr) return fail(PGG_ERR_NULL, "pointer is NULL");
    static_assert(sizeof(cudaIpcMemHandle_t) == PGG_SLAB_IPC_HANDLE_BYTES, "IPC handle size");
    cudaIpcMemHandle_t h;
    PGG_CUDA(cudaIpcGetMemHandle(&h, d_ptr));
    std::memcpy(h_handle64, &h, sizeof h);
    return PGG_OK;
}

int32_t pgg_slab_ipc_open(const uint8_t* h_handle64, int32_t peer_device, void** d_out)
{
    if (h_handle64 == nullptr || d_out == nullptr) return fail(PGG_ERR_NULL, "pointer is NULL");
    int dev = -1;
    PGG_CUDA(cudaGetDevice(&dev));
    if (peer_device >= 0 && peer_device != dev) {
        int can = 0;
        PGG_CUDA(cudaDeviceCanAccessPeer(&can, dev, peer_device));
        if (!can) return fail(PGG_ERR_UNSUPPORTED, "device %d cannot access device %d (no P2P path)", dev, peer_device);
        cudaError_t e = cudaDeviceEnablePeerAccess(peer_device, 0);
        if (e == cudaErrorPeerAccessAlreadyEnabled) (void)cudaGetLastError();
        else if (e != cudaSuccess) return fail(PGG_ERR_CUDA, "cudaDeviceEnablePeerAccess(%d) failed: %s", peer_device, cudaGetErrorString(e));
    }
    cudaIpcMemHandle_t h;
    std::memcpy(&h, h_handle64, sizeof h);
    void* p = nullptr;
    PGG_CUDA(cudaIpcOpenMemHandle(&p, h, cudaIpcMemLazyEnablePeerAccess));
    *d_out = p;
    return PGG_OK;
}

int32_t pgg_slab_ipc_close(void* d_ptr)
{
    if (d_ptr != nullptr) PGG_CUDA(cudaIpcCloseMemHandle(d_ptr));
    return PGG_OK;
}

int32_t pgg_trim_workspace(void)
{
    int dev = -1;
    PGG_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(PGG_ERR_UNSUPPORTED, "device ordinal %d", dev);
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    if (g_pool[dev] != nullptr) PGG_CUDA(cudaMemPoolTrimTo(g_pool[dev], 0));
    return PGG_OK;
}

uint64_t pgg_launch_count(void) { return g_launches.load(); }

const char* pgg_last_error(void) { return g_last_error.c_str(); }

}  // extern "C"
