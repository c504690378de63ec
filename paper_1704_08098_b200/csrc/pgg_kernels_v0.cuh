// pgg_kernels_v0.cuh -- support kernels (init, density, phase-class draw, count
// finalisation) and the V0 phase kernel: one thread per active site, plain
// global loads with periodic wrap.  V0 is the general path (any L % 4 == 0,
// both layouts) and the rung every faster variant is checked against.
#pragma once
#include "pgg_common.cuh"

namespace pgg {

// ---------------------------------------------------------------------------
// Per-lattice parameters (seed, acceptance table) travel to the device as KERNEL ARGUMENTS of
// this little kernel, five lattices per launch: no copy from pageable host memory, so no entry
// point ever waits for the stream, the caller's host arrays may die on return, and the calls can
// be captured into a CUDA graph.
// ---------------------------------------------------------------------------
constexpr int kParamPackLattices = 5;  // 5 x (8 + 612) bytes + header < the 4 KB argument limit
struct ParamPack {
    uint32_t n;                                     // lattices in this pack
    uint32_t with_tables;
    uint64_t seeds[kParamPackLattices];
    uint32_t tables[kParamPackLattices * kTableSize];
};

__global__ void __launch_bounds__(256)
upload_params_kernel(const __grid_constant__ ParamPack p, uint32_t first, uint64_t* __restrict__ seeds,
                     uint32_t* __restrict__ tables)
{
    if (threadIdx.x < p.n) seeds[first + threadIdx.x] = p.seeds[threadIdx.x];
    if (p.with_tables)
        for (uint32_t q = threadIdx.x; q < p.n * kTableSize; q += blockDim.x)
            tables[(size_t)first * kTableSize + q] = p.tables[q];
}

// ---------------------------------------------------------------------------
// K0 init: s(site) = [x0 < thr], x0 = word 0 of
// Philox(ctr = (site,0,0,INIT), key = seed), thr = floor(rho0 * 2^32) in [0, 2^32].
// u8: one thread writes 16 consecutive sites (one 16-byte store).
// bits: one thread writes one 32-site word.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
init_u8_kernel(uint8_t* __restrict__ lats, unsigned long long lat_bytes,
               const uint64_t* __restrict__ seeds, uint32_t n_sites, unsigned long long thr)
{
    const uint32_t b = blockIdx.y;
    const uint64_t seed = seeds[b];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    uint8_t* lat = lats + (size_t)b * lat_bytes;
    const uint32_t n_chunks = n_sites >> 4;  // L % 4 == 0  =>  L*L % 16 == 0
    for (uint32_t q = blockIdx.x * blockDim.x + threadIdx.x; q < n_chunks;
         q += gridDim.x * blockDim.x) {
        uint32_t w[4] = {0u, 0u, 0u, 0u};
#pragma unroll
        for (int a = 0; a < 16; ++a) {
            uint32_t x[4];
            philox4x32_10(q * 16u + a, 0u, 0u, kTagInit, k0, k1, x);
            const uint32_t s = ((unsigned long long)x[0] < thr) ? 1u : 0u;
            w[a >> 2] |= s << (8 * (a & 3));
        }
        reinterpret_cast<uint4*>(lat)[q] = make_uint4(w[0], w[1], w[2], w[3]);
    }
}

__global__ void __launch_bounds__(256)
init_bits_kernel(uint8_t* __restrict__ lats, unsigned long long lat_bytes,
                 const uint64_t* __restrict__ seeds, uint32_t n_sites, unsigned long long thr)
{
    const uint32_t b = blockIdx.y;
    const uint64_t seed = seeds[b];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    uint32_t* lat = reinterpret_cast<uint32_t*>(lats + (size_t)b * lat_bytes);
    const uint32_t n_words = n_sites >> 5;
    for (uint32_t q = blockIdx.x * blockDim.x + threadIdx.x; q < n_words;
         q += gridDim.x * blockDim.x) {
        uint32_t w = 0u;
#pragma unroll 8
        for (int a = 0; a < 32; ++a) {
            uint32_t x[4];
            philox4x32_10(q * 32u + a, 0u, 0u, kTagInit, k0, k1, x);
            w |= (((unsigned long long)x[0] < thr) ? 1u : 0u) << a;
        }
        lat[q] = w;
    }
}

// ---------------------------------------------------------------------------
// K3 density (Eq. 4): cooperator count of each lattice.
// 16-byte loads, popcount (u8 cells hold 0/1, so popc(word & 0x01010101) is
// the sum of the four bytes), warp redux, one 64-bit atomic per CTA.
// out[b * out_stride] must be zero on entry.
// ---------------------------------------------------------------------------
template <int FMT>
__global__ void __launch_bounds__(256)
density_kernel(const uint8_t* __restrict__ lats, unsigned long long lat_bytes,
               unsigned long long* __restrict__ out, uint32_t out_stride)
{
    const uint32_t b = blockIdx.y;
    const uint4* p = reinterpret_cast<const uint4*>(lats + (size_t)b * lat_bytes);
    const size_t n16 = lat_bytes >> 4;
    const uint32_t mask = (FMT == kFmtU8) ? 0x01010101u : 0xFFFFFFFFu;
    unsigned int acc = 0;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n16;
         q += (size_t)gridDim.x * blockDim.x) {
        const uint4 v = __ldg(p + q);
        acc += __popc(v.x & mask) + __popc(v.y & mask) + __popc(v.z & mask) + __popc(v.w & mask);
    }
    // bits layout of a lattice smaller than 16 bytes (L = 4, 8 cannot be bits: L % 32 == 0)
    acc = __reduce_add_sync(0xFFFFFFFFu, acc);
    __shared__ unsigned int part[8];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long s = 0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += part[w];
        if (s) atomicAdd(out + (size_t)b * out_stride, s);
    }
}

// ---------------------------------------------------------------------------
// a1 phase-class draw: w[4q+m] = word m of
// Philox(ctr = (t,0,q,ORDER), key = seed), q = 0..3.
// IID : class of phase k = w[k] >> 28.
// PERM: classes sorted ascending by (w[c], c); phase k takes the k-th.
// One thread per (lattice b, MCS m of the chunk); writes 16 bytes.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
order_kernel(const uint64_t* __restrict__ seeds, uint32_t B, uint32_t t0, uint32_t n_chunk,
             uint32_t order_stride, int order_mode, uint8_t* __restrict__ order)
{
    const uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= B * n_chunk) return;
    const uint32_t b = idx / n_chunk, m = idx - b * n_chunk;
    const uint64_t seed = seeds[b];
    uint32_t w[16];
#pragma unroll
    for (uint32_t q = 0; q < 4; ++q)
        philox4x32_10(t0 + m, 0u, q, kTagOrder, (uint32_t)seed, (uint32_t)(seed >> 32), &w[4 * q]);
    uint32_t packed[4] = {0u, 0u, 0u, 0u};  // 16 classes, one byte each
    if (order_mode == 0) {
#pragma unroll
        for (int k = 0; k < 16; ++k) packed[k >> 2] |= (w[k] >> 28) << (8 * (k & 3));
    } else {
        // rank of class c = number of classes that sort before it
#pragma unroll
        for (int c = 0; c < 16; ++c) {
            int rank = 0;
#pragma unroll
            for (int d = 0; d < 16; ++d)
                rank += (w[d] < w[c] || (w[d] == w[c] && d < c)) ? 1 : 0;
#pragma unroll
            for (int q = 0; q < 4; ++q)  // phase `rank` visits class c
                if ((rank >> 2) == q) packed[q] |= (uint32_t)c << (8 * (rank & 3));
        }
    }
    reinterpret_cast<uint4*>(order)[(size_t)b * order_stride + m] =
        make_uint4(packed[0], packed[1], packed[2], packed[3]);
}

// ---------------------------------------------------------------------------
// a8 trace: counts[b][m] = count0[b] + sum_{m' <= m} delta[b][m'],
// in place over the delta row.  One CTA per lattice; each thread scans a
// contiguous slice, the slice totals are scanned through shared memory.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(1024)
finalize_counts_kernel(unsigned long long* __restrict__ counts, uint32_t n_mcs,
                       const unsigned long long* __restrict__ count0)
{
    const uint32_t b = blockIdx.x;
    unsigned long long* row = counts + (size_t)b * n_mcs;
    const uint32_t per = (n_mcs + blockDim.x - 1) / blockDim.x;
    const uint32_t lo = min(threadIdx.x * per, n_mcs), hi = min(lo + per, n_mcs);
    unsigned long long s = 0;
    for (uint32_t m = lo; m < hi; ++m) s += row[m];
    __shared__ unsigned long long tot[1024];
    tot[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long run = count0[b];
        for (uint32_t a = 0; a < blockDim.x; ++a) {
            const unsigned long long v = tot[a];
            tot[a] = run;
            run += v;
        }
    }
    __syncthreads();
    unsigned long long run = tot[threadIdx.x];
    for (uint32_t m = lo; m < hi; ++m) {
        run += row[m];
        row[m] = run;
    }
}

// ---------------------------------------------------------------------------
// V0 phase kernel (steps a3-a8 of section 8(a)).
// Thread a < (L/4)^2 owns the active site (4*(a / (L/4)) + ci, 4*(a % (L/4)) + cj).
// Race-free in place (S1): the step reads only sites within Manhattan distance
// 3 of x, other active sites are >= 4 away, and it writes only x.
// ---------------------------------------------------------------------------
template <int FMT, int GAME = kGamePGG>
__global__ void __launch_bounds__(256)
phase_v0_kernel(PhaseArgs a, uint32_t m, uint32_t k)
{
    const uint32_t b = blockIdx.y;
    const uint32_t cls = a.order[((size_t)b * a.order_stride + (m % a.order_stride)) * 16 + k];
    const int ci = (int)(cls >> 2), cj = (int)(cls & 3u);
    const StepKey sk = make_step_key(a.seeds[b], a.t_begin + m, k, cls);
    const uint32_t* __restrict__ table = a.tables + (size_t)b * kTableSize;
    Lattice<FMT> lat{a.lats + (size_t)b * a.lat_bytes, (int)a.L};
    const int L = (int)a.L, m4 = L >> 2;
    const uint32_t n_cls = (uint32_t)m4 * (uint32_t)m4;
    const uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x;
    int delta = 0;
    if (idx < n_cls) {
        const int bi = (int)(idx / (uint32_t)m4), bj = (int)(idx - (uint32_t)bi * (uint32_t)m4);
        const int i = 4 * bi + ci, j = 4 * bj + cj;
        const int sx = lat.get(i, j);
        const int s_up = lat.get(i - 1, j), s_dn = lat.get(i + 1, j);
        const int s_lf = lat.get(i, j - 1), s_rt = lat.get(i, j + 1);
        // S9: if all four neighbours share s_x no draw can change the state
        if (s_up + s_dn + s_lf + s_rt != 4 * sx) {
            uint32_t x0, u;
            step_draw(sk, (uint32_t)i * (uint32_t)L + (uint32_t)j, x0, u);
            const int dir = (int)(x0 >> 30);  // 0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1)
            const int sy = dir == 0 ? s_up : dir == 1 ? s_dn : dir == 2 ? s_lf : s_rt;
            if (sy != sx) {
                const int yi = i + (dir == 0 ? -1 : dir == 1 ? 1 : 0);
                const int yj = j + (dir == 2 ? -1 : dir == 3 ? 1 : 0);
                // public goods game: the difference of the integer payoffs A; prisoner's dilemma
                // (PAPER.md:131): the cooperating neighbours of x and of y, radius 2 only
                const int idx_t = GAME == kGamePD
                                      ? sx * 25 + (s_up + s_dn + s_lf + s_rt) * 5 + pd_neighbour_count(lat, yi, yj)
                                      : table_index(payoff_A(lat, i, j) - payoff_A(lat, yi, yj), sx - sy);
                if (u < table[idx_t]) {
                    lat.flip_to(i, j, sy);
                    delta = sy - sx;
                }
            }
        }
    }
    if (a.deltas != nullptr) {
        delta = __reduce_add_sync(0xFFFFFFFFu, delta);
        __shared__ int part[8];
        if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = delta;
        __syncthreads();
        if (threadIdx.x == 0) {
            int s = 0;
            for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += part[w];
            if (s != 0)
                atomicAdd(a.deltas + (size_t)b * a.n_mcs + m, (unsigned long long)(long long)s);
        }
    }
}

}  // namespace pgg
