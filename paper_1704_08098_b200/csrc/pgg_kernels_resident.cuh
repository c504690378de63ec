// pgg_kernels_resident.cuh -- the RESIDENT sweep kernel (K4 for small lattices, both layouts).
//
// For L <= 512 a phase touches so few sites that the per-phase launches of the streaming
// kernels are latency-bound (measured: 4-30 us per launch against < 1 us of work, DESIGN.md
// section 6).  Here ONE CTA per lattice keeps the whole lattice in shared memory, bit-packed
// with a 3-site periodic ghost frame, and runs every phase of every MCS of the call without
// leaving the SM: 16 * n_mcs launches become one (per chunk of <= 4096 MCS, the length of the
// phase-order buffer).
//
//   smem lattice : rows r = i + 3 in [0, L + 6), columns c = j + 3 in [0, L + 6); site (r, c) is
//                  bit (c & 31) of word r * PW + (c >> 5).  The frame holds the periodic images,
//                  so a stencil read is bits[off + constant]: no wrap arithmetic.  A flip also
//                  flips its images (sites within 3 of an edge).
//   phase, pass 1: word-parallel S9 bulk test of the active rows (32 sites per word op, as the
//                  bit-packed streaming kernels do); surviving sites go to a CTA-wide list
//                  (warp prefix sum + one shared atomic per warp).
//   phase, pass 2: the list is processed densely, one site per thread: Philox draw (a3),
//                  neighbour compare (a4), 14-read stencil A_x - A_y (a5), threshold compare (a6),
//                  atomicXor of the site's bit and its images (a7), signed flip count (a8).
//   In-place updates are race-free (S1): nothing within Manhattan distance 3 of an active site
//   is written in the same phase; the frame images of a site are read only by stencils that
//   may read the site itself.
#pragma once
#include "pgg_common.cuh"
#include "pgg_stencil_lut.cuh"

namespace pgg {

constexpr int kResThreads = 1024;
constexpr uint32_t kResMaxL = 512;

struct ResPlan {
    uint32_t PW;          // words per smem row = ceil((L + 6) / 32)
    uint32_t n_words;     // (L + 6) * PW
    uint32_t list_cap;    // (L / 4)^2 entries
    uint32_t smem_bytes;
};

inline bool resident_supported(int fmt, uint32_t L)
{
    if (L < 8 || L > kResMaxL || L % 4 != 0) return false;
    return fmt == kFmtU8 || L % 32 == 0;
}

__device__ __forceinline__ int res_get(const uint32_t* bits, int off)
{
    return (int)((bits[off >> 5] >> (off & 31)) & 1u);
}

template <int FMT>
__global__ void __launch_bounds__(kResThreads, 1)
sweep_resident_kernel(PhaseArgs a, uint32_t m0, uint32_t n_chunk, ResPlan g)
{
    extern __shared__ __align__(16) uint32_t res_smem[];
    uint32_t* bits = res_smem;
    uint32_t* list = bits + g.n_words;            // (r << 16) | c of the sites that need a draw
    uint32_t* tbl = list + g.list_cap;
    const int8_t* lut = reinterpret_cast<const int8_t*>(tbl + 160);  // StencilLut: the frame means no window ever wraps
    __shared__ uint32_t n_list[2];  // by phase parity: reset one while the other is in use
    __shared__ int s_delta[2];

    const uint32_t b = blockIdx.x;
    const int L = (int)a.L, PW = (int)g.PW, PB = 32 * PW;
    const int tid = threadIdx.x, lane = tid & 31;
    uint8_t* lat = a.lats + (size_t)b * a.lat_bytes;
    Lattice<FMT> glat{lat, L};

    // ---- load: every smem bit (r, c) <- s((r - 3) mod L, (c - 3) mod L)
    for (uint32_t q = tid; q < g.n_words; q += kResThreads) {
        const int r = (int)(q / (uint32_t)PW), c0 = 32 * (int)(q - (uint32_t)r * PW);
        int i = r - 3;
        i = i < 0 ? i + L : (i >= L ? i - L : i);
        uint32_t w = 0;
        for (int t = 0; t < 32; ++t) {
            const int c = c0 + t;
            if (c < L + 6) {
                int j = c - 3;
                j = j < 0 ? j + L : (j >= L ? j - L : j);
                w |= (uint32_t)glat.get(i, j) << t;
            }
        }
        bits[q] = w;
    }
    for (int q = tid; q < kTableSize; q += kResThreads) tbl[q] = a.tables[(size_t)b * kTableSize + q];
    for (int q = tid; q < kStencilLutBytes / 4; q += kResThreads)
        (tbl + 160)[q] = reinterpret_cast<const uint32_t*>(g_stencil_lut.v)[q];
    if (tid == 0) {
        n_list[0] = n_list[1] = 0u;
        s_delta[0] = s_delta[1] = 0;
    }
    __syncthreads();

    StepKey sk = make_step_key(a.seeds[b], 0u, 0u, 0u);  // round keys: functions of the seed only
    const int m4 = L >> 2;                 // active rows (and columns) per class
    const int n_rowwords = m4 * PW;        // word tasks of pass 1

    for (uint32_t mm = 0; mm < n_chunk; ++mm) {
        const uint32_t m = m0 + mm;
        // the 16 phase classes of this MCS: one 16-byte load
        const uint4 ord4 = *reinterpret_cast<const uint4*>(
            a.order + ((size_t)b * a.order_stride + (m % a.order_stride)) * 16);
        int delta = 0;
#pragma unroll 1
        for (uint32_t k = 0; k < 16; ++k) {
            const uint32_t ow = k < 8u ? (k < 4u ? ord4.x : ord4.y) : (k < 12u ? ord4.z : ord4.w);
            const uint32_t cls = (ow >> (8u * (k & 3u))) & 0xFFu;
            const int ci = (int)(cls >> 2), cj = (int)(cls & 3u);
            {   // only the site-independent half of round 1 depends on (t, k, class)
                const uint64_t p1 = (uint64_t)kPhiloxM1 * ((k << 8) | cls);
                sk.r1_c0 = (uint32_t)(p1 >> 32) ^ (a.t_begin + m) ^ sk.k0[0];
                sk.r1_c1 = (uint32_t)p1;
            }
            // ---- pass 1: S9 bulk test, 32 sites per word; active columns are c = 4 q + cj + 3
            const uint32_t cm = 0x11111111u << ((cj + 3) & 3);
            for (int base = 0; base < n_rowwords; base += kResThreads) {
                const int q = base + tid;
                uint32_t nb = 0;
                int r = 0, wq = 0;
                if (q < n_rowwords) {
                    const int ar = q / PW;
                    wq = q - ar * PW;
                    r = 4 * ar + ci + 3;
                    const uint32_t* row = bits + r * PW;
                    const uint32_t x = row[wq], up = row[wq - PW], dn = row[wq + PW];
                    const uint32_t pv = wq > 0 ? row[wq - 1] : 0u, nx = wq + 1 < PW ? row[wq + 1] : 0u;
                    const uint32_t lw = __funnelshift_l(pv, x, 1), rw = __funnelshift_r(x, nx, 1);
                    // valid columns of this word: 3 <= c < L + 3
                    const int lo = max(3 - 32 * wq, 0), hi = min(L + 3 - 32 * wq, 32);
                    uint32_t valid = 0u;
                    if (hi > lo) valid = (hi == 32 ? 0xFFFFFFFFu : ((1u << hi) - 1u)) & ~((1u << lo) - 1u);
                    nb = ((x ^ up) | (x ^ dn) | (x ^ lw) | (x ^ rw)) & cm & valid;  // S9
                }
                // warp prefix sum of the per-lane counts, one shared atomic per warp
                const int cnt = __popc(nb);
                int incl = cnt;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const int v = __shfl_up_sync(0xFFFFFFFFu, incl, d);
                    if (lane >= d) incl += v;
                }
                const int total = __shfl_sync(0xFFFFFFFFu, incl, 31);
                uint32_t at = 0;
                if (total) {
                    if (lane == 31) at = atomicAdd(&n_list[k & 1u], (uint32_t)total);
                    at = __shfl_sync(0xFFFFFFFFu, at, 31) + (uint32_t)(incl - cnt);
                    while (nb) {
                        const int bit = __ffs(nb) - 1;
                        nb &= nb - 1u;
                        list[at++] = ((uint32_t)r << 16) | (uint32_t)(32 * wq + bit);
                    }
                }
            }
            __syncthreads();
            // ---- pass 2: one listed site per thread
            const uint32_t nl = n_list[k & 1u];
            if (tid == 0) n_list[(k + 1u) & 1u] = 0u;  // last read before the previous barrier, next used after the next
            for (uint32_t q = tid; q < nl; q += kResThreads) {
                const uint32_t e = list[q];
                const int r = (int)(e >> 16), c = (int)(e & 0xFFFFu);
                const int i = r - 3, j = c - 3;
                const int off = r * PB + c;
                uint32_t x0, u;
                step_draw(sk, (uint32_t)i * (uint32_t)L + (uint32_t)j, x0, u);
                const uint32_t dir = x0 >> 30;  // 0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1)
                const int sx = res_get(bits, off);
                // bit offsets: e = step towards y, f = perpendicular step
                const int ee = dir < 2u ? (dir == 0u ? -PB : PB) : (dir == 2u ? -1 : 1);
                if (res_get(bits, off + ee) != sx) {
                    // A_x - A_y: six 7-bit windows (rows of the frame never wrap) index the weight table
                    const int dA = bits_stencil_lut(off, dir, sx, bits, PW, lut);
                    if (u < tbl[sx * 102 + dA + 25]) {
                        // flip the site and its frame images
                        const int r2 = i < 3 ? r + L : (i >= L - 3 ? r - L : -1);
                        const int c2 = j < 3 ? c + L : (j >= L - 3 ? c - L : -1);
                        atomicXor(bits + (off >> 5), 1u << (off & 31));
                        if (r2 >= 0) { const int o = r2 * PB + c; atomicXor(bits + (o >> 5), 1u << (o & 31)); }
                        if (c2 >= 0) { const int o = r * PB + c2; atomicXor(bits + (o >> 5), 1u << (o & 31)); }
                        if (r2 >= 0 && c2 >= 0) { const int o = r2 * PB + c2; atomicXor(bits + (o >> 5), 1u << (o & 31)); }
                        delta += 1 - 2 * sx;
                    }
                }
            }
            __syncthreads();
        }
        // ---- a8: signed flip count of this MCS (double-buffered accumulator)
        if (a.deltas != nullptr) {
            delta = __reduce_add_sync(0xFFFFFFFFu, delta);
            if (lane == 0 && delta != 0) atomicAdd(&s_delta[mm & 1u], delta);
            __syncthreads();
            if (tid == 0) {
                a.deltas[(size_t)b * a.n_mcs + m] = (unsigned long long)(long long)s_delta[mm & 1u];
                s_delta[mm & 1u] = 0;
            }
        }
    }
    __syncthreads();

    // ---- write back the core sites in the canonical layout
    if (FMT == kFmtU8) {
        const int n4 = L * (L >> 2);  // 4 sites per thread step
        for (int q = tid; q < n4; q += kResThreads) {
            const int i = q / (L >> 2), j = 4 * (q - i * (L >> 2));
            const int off = (i + 3) * PB + j + 3;
            uint32_t w = 0;
#pragma unroll
            for (int t = 0; t < 4; ++t) w |= (uint32_t)res_get(bits, off + t) << (8 * t);
            reinterpret_cast<uint32_t*>(lat)[q] = w;
        }
    } else {
        const int nw = L * (L >> 5);
        for (int q = tid; q < nw; q += kResThreads) {
            const int i = q / (L >> 5), j = 32 * (q - i * (L >> 5));
            const int off = (i + 3) * PB + j + 3;
            // 32 sites starting at smem bit `off` (off & 31 == 3): two words funnel-shifted
            const uint32_t w0 = bits[off >> 5], w1 = bits[(off >> 5) + 1];
            reinterpret_cast<uint32_t*>(lat)[q] = __funnelshift_r(w0, w1, off & 31);
        }
    }
}

inline int resident_plan(int fmt, uint32_t L, ResPlan* p)
{
    bool attr_set = false;  // per call (the function attribute is per device)
    p->PW = (L + 6 + 31) / 32;
    p->n_words = (L + 6) * p->PW;
    p->list_cap = (L / 4) * (L / 4);
    p->smem_bytes = (p->n_words + p->list_cap + 160) * 4 + kStencilLutBytes + 8;  // + 8: the window's second word after the last row
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(sweep_resident_kernel<kFmtU8>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e != cudaSuccess) return (int)e;
        e = cudaFuncSetAttribute(sweep_resident_kernel<kFmtBits>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 200 * 1024);
        if (e != cudaSuccess) return (int)e;
        attr_set = true;
    }
    (void)fmt;
    return 0;
}

inline void resident_launch(const ResPlan& p, int fmt, const PhaseArgs& a, uint32_t m0, uint32_t n_chunk,
                            uint32_t B, cudaStream_t stream)
{
    if (fmt == kFmtU8)
        sweep_resident_kernel<kFmtU8><<<B, kResThreads, p.smem_bytes, stream>>>(a, m0, n_chunk, p);
    else
        sweep_resident_kernel<kFmtBits><<<B, kResThreads, p.smem_bytes, stream>>>(a, m0, n_chunk, p);
}

}  // namespace pgg
