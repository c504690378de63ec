/*
 * pgg.h -- C ABI of libpgg: the Monte Carlo sweep of the spatial public goods
 * game (Perc, arXiv:1704.08098) on an L x L periodic square lattice, run under
 * the race-free 16-sublattice Philox schedule, as hand-written CUDA for sm_100a.
 *
 * Citations are "PAPER.md:<line>" (the paper's text, /root/reference/PAPER.md)
 * and "SURVEY 8(c) Dn/Sn" (the readings listed in SURVEY.md section 8(c) and
 * restated in DESIGN.md).  Everything the method computes runs in CUDA kernels
 * of this library; there is no CPU fallback.  Every entry point returns
 * PGG_OK (0) or a negative PGG_ERR_* code; nothing is printed, no exception
 * crosses the boundary.  pgg_last_error() gives a thread-local text.
 *
 * Model.  s(i,j) in {0,1}: D = 0, C = 1.  cross(z) = z and its
 * four nearest neighbours (the von Neumann group centred on z, G = 5).
 * N(z) = number of cooperators in cross(z).  A_x = sum of N(z) over the five
 * groups z in cross(x) that player x belongs to.  With c = 1 (Eqs. 1-2,
 * PAPER.md:47-50) the total payoff is  Pi_x = (r/5) A_x - 5 s_x.
 * Elementary step: focal x, random nearest neighbour y, x adopts
 * s_y with W = 1/(1+exp((Pi_x-Pi_y)/K))  (Eq. 3).
 *
 * Schedule (north_star).  class(i,j) = 4*(i mod 4) +
 * (j mod 4).  One MCS t = 16 phases k = 0..15; phase k updates, in place and
 * all at once, every site of one class c(t,k) drawn from Philox4x32-10; each
 * site draws (direction, u) from Philox4x32-10 with counter
 * (site, t, (k<<8)|c, 3) and key (seed lo, seed hi); x adopts s_y iff
 * s_x != s_y and u < T[(s_x-s_y+1)*51 + (A_x-A_y+25)].
 *
 * Pointers named d_* are DEVICE pointers, h_* are HOST pointers.  The caller
 * owns every buffer.  `stream` is a cudaStream_t passed as void* (NULL = the
 * legacy default stream).  All device work is enqueued on `stream`; no entry
 * point waits for the stream or the device (pgg_phase_classes, which returns host data, is the one
 * exception and says so): per-lattice parameters reach the device as kernel arguments, not by
 * copies from pageable memory, so host arrays may be freed on return.  Results are valid once
 * the caller has synchronised the stream.  The kernel-variant switch (pgg_set_variant) and the
 * environment knobs DESIGN.md lists are process-wide; a call uses the current CUDA device.
 * Temporary device memory (seeds, tables, class order, the working copy of PGG_VARIANT_PACKED) is taken
 * from and returned to a stream-ordered memory pool the library owns, one per device
 * (cudaMallocFromPoolAsync / cudaFreeAsync; pgg_trim_workspace() gives it back to the driver);
 * pgg_sweep_static takes none at all.
 */
#ifndef PGG_H_
#define PGG_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    PGG_OK = 0,
    PGG_ERR_NULL = -1,        /* a required pointer is NULL                              */
    PGG_ERR_BAD_L = -2,       /* L < 4, L % 4 != 0, L >= 65536 (site indices are uint32: every
                                 entry point, pgg_density included), or (bits) L % 32 != 0 */
    PGG_ERR_BAD_PARAM = -3,   /* r/K not finite, K <= 0, rho0 outside [0,1], B == 0, ... */
    PGG_ERR_ALIGN = -4,       /* lattice pointer not 16-byte aligned                     */
    PGG_ERR_UNSUPPORTED = -5, /* unknown fmt / order_mode / kernel variant               */
    PGG_ERR_CUDA = -6         /* a CUDA runtime call failed; see pgg_last_error()        */
};

/* Canonical lattice layouts.
 * PGG_FMT_U8  : row-major uint8 [L][L], 1 = C, 0 = D.  Any L with L % 4 == 0.
 * PGG_FMT_BITS: row-major, site (i,j) is bit (j & 31) of the little-endian uint32
 *               word i*(L/32) + (j >> 5).  Needs L % 32 == 0.                    */
enum { PGG_FMT_U8 = 0, PGG_FMT_BITS = 1 };

/* How the 16 phase classes of an MCS are drawn.
 * PGG_ORDER_IID : class of phase k = top 4 bits of word k (default; reproduces
 *                 random-sequential statistics).
 * PGG_ORDER_PERM: a permutation -- classes sorted by (word[c], c).
 * PGG_ORDER_DTILE: not a class order but the paper's own schedule, the double
 *   tiling decomposition (Fig. 2): 4x4 domains, domain (I,J) =
 *   (i>>2, j>>2) of type 2*(I&1) + (J&1), L % 8 == 0; one MCS =
 *   four parts, types 0,1,2,3 in turn; in a part every domain of
 *   the type makes 16 sequential elementary steps on its own sites (so that an
 *   MCS is L^2 steps); pick p of domain d = I*(L/4) + J in MCS t
 *   draws (x0,x1,x2,.) = Philox4x32-10(ctr = (d, t, p, 5), key = seed): focal
 *   site = domain row x0>>30, domain column (x0>>28)&3, neighbour direction
 *   x2>>30 (0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1)), u = x1; x adopts s_y iff
 *   s_x != s_y and u < T[...] as in every mode.  Kernel variants do not apply. */
enum { PGG_ORDER_IID = 0, PGG_ORDER_PERM = 1, PGG_ORDER_DTILE = 2 };

/* Kernel variants of the phase step (all bit-identical).
 * PGG_VARIANT_AUTO picks by measurement (DESIGN.md appendix B): CLUSTER for L = 512 and 1024 and for
 * L = 2048 from 32 lattices; else RESIDENT for L <= 320 and for L <= 448 from 3 lattices; else, for
 * L = 1024 .. 32768 (powers of two), LEAN for the bit-packed layout and PACKED (a bit-packed working copy +
 * LEAN) for uint8 from L = 2048; else RING (uint8) / BAND (bit-packed) for
 * L >= 2048 and for uint8 L = 512; else V0.  TILE, PIPE, SPLIT, DYN, BAND (uint8), PERSIST are rungs of the
 * ladder kept for comparison: selectable, tested, never chosen.  Tuning knobs read from the environment by
 * the plan functions (defaults are the measured best; every setting is bit-exact): PGG_PDL,
 * PGG_RING_{SLOTS,L2PF,FULLROW,TPR_LOG2,MIRROR,ROTATE}, PGG_BAND_SLOTS, PGG_DYN_WARPS, PGG_PIPE_STAGES,
 * PGG_TILE_{CTAS_PER_SM,STAGES}, PGG_LEAN_{LAG,AHEAD,SLOT_ROWS,SLOTS,WORDS}, PGG_CLUSTER_SIZE, and
 * PGG_PACKED_MIN_L (the smallest uint8 L for which AUTO takes PACKED; read once per process).             */
enum {
    PGG_VARIANT_AUTO = 0,
    PGG_VARIANT_V0 = 1,   /* one thread per active site, global loads, any L % 4 == 0 */
    PGG_VARIANT_TILE = 2, /* smem tile + 3-site halo, bulk-async staged, compaction   */
    /* 3 is unused (a temporal-blocking variant was never built: DESIGN.md section 9)   */
    PGG_VARIANT_PIPE = 4, /* TILE staging as a producer/consumer warp pipeline        */
    PGG_VARIANT_BAND = 5, /* row bands of wide strips streamed through a smem ring    */
    PGG_VARIANT_RING = 6, /* BAND's data movement, consumer cut to the fewest instr.  */
    PGG_VARIANT_SPLIT = 7,/* RING with scanner and worker warps (uint8 only)          */
    PGG_VARIANT_DYN = 8,  /* RING with dynamically assigned tasks, 24 warps (uint8)   */
    PGG_VARIANT_RESIDENT = 9,/* L <= 512: one CTA per lattice, lattice resident in smem,
                                every phase of the call in one launch                  */
    PGG_VARIANT_DTILE = 10,  /* reported by pgg_get_variant_used() after a PGG_ORDER_DTILE
                                sweep (one thread per 4x4 domain); not selectable       */
    PGG_VARIANT_LEAN = 11,   /* L = 1024 .. 32768, a power of two: whole rows streamed, packed to
                                bits on arrival (uint8), scan / draw / stencil on a bit ring   */
    PGG_VARIANT_PERSIST = 12,/* LEAN, bit-packed, <= 148 lattices: every phase of up to 4096 MCS in ONE
                                cooperative launch; between phases a band waits for its two neighbour bands only */
    PGG_VARIANT_CLUSTER = 13,/* L = 128 .. 4096 (a power of two), both layouts: the lattice stays bit-packed in
                                the shared memory of a CTA cluster (1 .. 16 CTAs) for the whole call; after a phase
                                the changed halo row goes to each neighbour over distributed shared memory by
                                asynchronous stores that complete on the neighbour's mbarrier (no cluster barrier) */
    PGG_VARIANT_PACKED = 14  /* uint8 lattices, L = 1024 .. 32768 (a power of two): the call packs the lattice
                                into a bit-packed WORKING COPY (L*L/8 bytes per lattice from the stream-ordered
                                pool: 32 MiB at L = 16384, which stays in the 126 MB L2), runs every phase on
                                it with LEAN, and unpacks it into the caller's uint8 lattice when the call ends
                                (the internal layout SURVEY 8(b) allows behind the canonical ones).  The
                                caller's lattice holds the result when the call's work on the stream is done,
                                as always; while the call runs it holds the state the call started from.  */
};

/* Acceptance table, Eq. (3) PAPER.md:60 in the integer form of SURVEY 8(c) D3:
 * for ds in {-1,0,1}, dA in [-25,25], in IEEE double and in this order,
 *   delta = (r*dA)/5 - 5*ds;  W = 1/(1+exp(delta/K));  v = W * 2^32;
 *   T = v >= 4294967295 ? 0xFFFFFFFF : (uint32)floor(v)
 * stored at out153[(ds+1)*51 + (dA+25)].  Pure host function (no CUDA call).
 * h_out153: host array of 153 uint32, written.
 * Errors: NULL -> PGG_ERR_NULL; r or K not finite, K <= 0 -> PGG_ERR_BAD_PARAM. */
int32_t pgg_build_accept_table(double r, double K, uint32_t* h_out153);

/* Initial condition ("C or D with equal probability"):
 * s(site) = [ x0 < floor(rho0 * 2^32) ], (x0,..) = Philox4x32-10(ctr = (site,0,0,1),
 * key = seed).  rho0 = 0 gives all D, rho0 = 1 all C, exactly.
 * d_lat: device lattice in layout `fmt`, L*L bytes (u8) or L*L/8 bytes (bits),
 * 16-byte aligned, overwritten.                                                  */
int32_t pgg_init_lattice(void* d_lat, int32_t fmt, uint32_t L, double rho0, uint64_t seed,
                         void* stream);

/* n_mcs full Monte Carlo steps t = t_begin .. t_begin+n_mcs-1 (1 MCS = L^2
 * elementary steps, PAPER.md:65 = 16 phases of L^2/16 sites), in place.
 * d_counts: NULL, or device array of n_mcs uint64; d_counts[m] = number of
 *   cooperators (numerator of Eq. 4) after MCS t_begin+m completes.
 * The RNG is counter based, so (t_begin=a, n=b) followed by (a+b, c) equals
 * (a, b+c) bit for bit.
 * Errors: PGG_ERR_NULL (d_lat), PGG_ERR_BAD_L, PGG_ERR_ALIGN, PGG_ERR_BAD_PARAM
 * (r, K not finite, K <= 0, t_begin + n_mcs > 2^32), PGG_ERR_UNSUPPORTED
 * (fmt, order_mode), PGG_ERR_CUDA.  n_mcs == 0 is a no-op.  PGG_ORDER_DTILE needs
 * L % 8 == 0, else PGG_ERR_BAD_L.                                   */
int32_t pgg_sweep(void* d_lat, int32_t fmt, uint32_t L, double r, double K, uint64_t seed,
                  int32_t order_mode, uint32_t t_begin, uint32_t n_mcs, uint64_t* d_counts,
                  void* stream);

/* pgg_sweep for callers that may not allocate (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): same operation, same arguments, same
 * results bit for bit (the 16-phase schedule of pgg_sweep), but the
 * temporaries of the sweep -- the seed, the 153-entry acceptance table (Eq. 3),
 * the initial cooperator count and the phase-class order of every MCS of the call (16 bytes
 * per MCS) -- live in ONE file-scope device array of PGG_STATIC_SCRATCH_BYTES (65 KB, held
 * by every GPU that loads the library until the process exits) instead of the stream-ordered
 * pool.  The call makes no cudaMalloc / cudaMallocAsync / cudaFree and calls no allocating
 * library routine; the caller still owns d_lat and d_counts.
 *   limit   : n_mcs <= PGG_STATIC_MAX_MCS (4096) per call, else PGG_ERR_BAD_PARAM (split a
 *             longer run into several calls: (t_begin = a, n = b) then (a + b, c) equals
 *             (a, b + c) bit for bit, as for pgg_sweep); PGG_ORDER_IID / PGG_ORDER_PERM only
 *             (PGG_ORDER_DTILE -> PGG_ERR_UNSUPPORTED).
 *   kernels : the one pgg_sweep would pick for a single lattice among CLUSTER, RESIDENT,
 *             LEAN, RING and V0 (pgg_set_variant is honoured for these five; any other
 *             selected variant -> PGG_ERR_UNSUPPORTED).
 *   sharing : every call on a device uses the same array and finds the previous call's
 *             contents in it; the call overwrites all it reads (and clears the one counter
 *             that must start at zero) in stream order.  Two calls that OVERLAP on the GPU
 *             (different streams without an event between them, or two host threads) race
 *             on the array: serialise them.  Calls on one stream are safe back to back.
 * Other errors as pgg_sweep.                                                         */
#define PGG_STATIC_MAX_MCS 4096u
#define PGG_STATIC_SCRATCH_BYTES (1024u + 16u * PGG_STATIC_MAX_MCS)
int32_t pgg_sweep_static(void* d_lat, int32_t fmt, uint32_t L, double r, double K, uint64_t seed,
                         int32_t order_mode, uint32_t t_begin, uint32_t n_mcs, uint64_t* d_counts,
                         void* stream);

/* Cooperator count sum_x d_x (Eq. 4; rho_C = count / L^2).
 * d_count: device uint64, overwritten.                                           */
int32_t pgg_density(const void* d_lat, int32_t fmt, uint32_t L, uint64_t* d_count, void* stream);

/* B independent lattices in one grid per phase (north_star (5)): lattice b has
 * its own r (h_r[b]) and seed (h_seeds[b]) and therefore its own acceptance
 * table, phase-class order and draws; it evolves exactly as a solo pgg_sweep
 * with (h_r[b], h_seeds[b]) would.
 * d_lats : B lattices, contiguous, each L*L bytes (u8) or L*L/8 bytes (bits).
 * h_r, h_seeds: host arrays of B entries, read before the call returns.
 * rho0   : in [0,1] -> first initialise lattice b by pgg_init_lattice(seed b);
 *          < 0 -> continue from the state given in d_lats.
 * d_counts: NULL or device array [B][n_mcs] uint64, as in pgg_sweep.             */
int32_t pgg_run_ensemble(void* d_lats, int32_t fmt, uint32_t B, uint32_t L, const double* h_r,
                         double K, const uint64_t* h_seeds, int32_t order_mode, double rho0,
                         uint32_t t_begin, uint32_t n_mcs, uint64_t* d_counts, void* stream);

/* ---- The prisoner's dilemma (section VI): "the described parallelization scheme can be
 * easily adapted so that ... other evolutionary games on the square lattice can be performed, such as
 * ... the well-known prisoner's dilemma game ... played in a pairwise manner, not in groups.  As a
 * consequence, the memory needed ... is one line outward less in each direction".  The paper gives no
 * payoff matrix; readings (G1-G4):
 *  G1 x plays one two-player game with each of its four nearest neighbours (not with itself); a pair
 *     earns C-C: R, C-D: S, D-C: T, D-D: P; Pi_x = the sum of its four games.  (R = 1, S = P = 0, T = b
 *     is the weak dilemma of the literature the paper cites.)
 *  G2 the elementary step, the Fermi rule (Eq. 3), the 16-sublattice schedule and the draws are those
 *     of pgg_sweep.
 *  G3 with n_z = cooperators among the four neighbours of z: Pi_z = s_z ? R n_z + S (4 - n_z)
 *     : T n_z + P (4 - n_z); thresholds T[s_x*25 + n_x*5 + n_y] for s_y = 1 - s_x, in IEEE double:
 *     z = (Pi_x - Pi_y)/K; W = 1/(1+exp(z)); v = W * 2^32; T = v >= 4294967295 ? 0xFFFFFFFF : floor(v).
 *  G4 a step reads within Manhattan distance 2 of x.
 * pgg_pd_build_accept_table: pure host function, h_out50 = 50 uint32.  pgg_pd_sweep: arguments and
 * errors as pgg_sweep with (R, S, T, P) in place of r; PGG_ORDER_IID / PGG_ORDER_PERM only; runs on the
 * LEAN kernel where it is supported (L = 1024 .. 32768, a power of two), else on V0.                    */
int32_t pgg_pd_build_accept_table(double R, double S, double T, double P, double K, uint32_t* h_out50);
int32_t pgg_pd_sweep(void* d_lat, int32_t fmt, uint32_t L, double R, double S, double T, double P, double K,
                     uint64_t seed, int32_t order_mode, uint32_t t_begin, uint32_t n_mcs, uint64_t* d_counts,
                     void* stream);

/* ---- One lattice sharded over several GPUs as ROW SLABS (the periodic L x L lattice
 * is PAPER.md:45, the step PAPER.md:58-60).  One process per GPU holds lattice rows [row0, row0 + n_rows)
 * plus three halo rows on either side -- the read stencil of a step has radius 3:
 *   d_slab : (n_rows + 6) whole rows in layout fmt (pgg_slab_bytes), 16-byte aligned; buffer row q holds
 *            lattice row (row0 - 3 + q) mod L.  The caller fills own rows AND halo rows once, before the
 *            first phase; after that the library keeps the halos current.
 *   row0 % 4 == 0, n_rows % 4 == 0, n_rows >= 4, row0 + n_rows <= L.
 * pgg_slab_sweep runs n_phases consecutive phases of the 16-sublattice schedule on the slab's own rows,
 * starting at phase k_begin (0..15) of MCS t_begin and running on into the following MCS.  The Philox
 * counter carries the site index of the WHOLE lattice, so the slabs together evolve bit for bit as
 * pgg_sweep evolves the unsharded lattice (r, K, seed, order_mode as there; PGG_ORDER_IID / _PERM only).
 * Halo push, fused into the phase kernel: a thread that flips a site of the slab's first (last) three own
 * rows also stores the new value through d_up_halo (d_dn_halo):
 *   d_up_halo : three rows, layout fmt -- the upper neighbour's copy of this slab's own rows 0..2, i.e. rows
 *               n_rows' + 3 .. n_rows' + 5 of ITS buffer (n_rows' = its row count);
 *   d_dn_halo : three rows -- the lower neighbour's copy of own rows n_rows-3 .. n_rows-1 = rows 0..2 of its buffer.
 *   Both are plain device pointers: memory of this GPU (several slabs on one device; a single slab is its own
 *   neighbour both ways) or of a peer GPU (pgg_slab_ipc_open; stores and 32-bit atomics over NVLink P2P).
 * Order between phases.  Phase p + 1 of a slab needs phase p of its two neighbours complete (their pushes
 * landed; and they have finished reading what p + 1 overwrites).  Two ways:
 *   d_flags == NULL : the caller orders the launches (slabs of one device driven phase by phase on one stream).
 *   d_flags != NULL : three uint32 on THIS device (zero before epoch 0): [0] internal, [1] / [2] = phases the
 *               upper / lower neighbour has completed.  d_up_flag = address of the upper neighbour's
 *               flags[2], d_dn_flag = address of the lower neighbour's flags[1] (local or peer memory).  The
 *               phase with global number e = epoch0 + p starts when flags[1] >= e and flags[2] >= e (acquire,
 *               system scope; a wait of seconds traps instead of hanging) and, complete, stores e + 1 to both
 *               neighbours (release, system scope).  All slabs of the lattice must run the same phases with the
 *               same epoch numbers; epoch0 continues from call to call.  No host synchronisation, no NCCL on
 *               the data path: neighbouring slabs are at most one phase apart.  ONE SLAB PER DEVICE when the flags
 *               are meant to wait: a waiting kernel holds its SMs, so two slabs of one device on different streams
 *               can starve each other until the wait traps.  Slabs that share a device are launched phase by phase
 *               in dependency order on one stream (every slab runs phase p before any runs p + 1); the flags are
 *               then always found set (paper_1704_08098_b200/slab.py: LocalSlabs).
 *   d_deltas : NULL or device array of uint64 (two's complement), one per MCS the call touches
 *               (ceil((k_begin + n_phases) / 16)): the signed number of flips of this slab's own rows in MCS
 *               t_begin + m is ADDED to d_deltas[m].  The rho_C trace (Eq. 4) is the initial count
 *               plus the running sum of the deltas summed over all slabs (one all-reduce per call, not per phase).
 * At most PGG_SLAB_MAX_MCS MCS per call.  Kernels: a slab of whole LEAN steps (L = 1024 .. 32768, a power of two;
 * row0 and n_rows multiples of pgg_slab_step_rows(fmt, L)) runs LEAN's ring kernel on the slab's buffer, and only
 * its first / last row band waits for and posts to the upper / lower neighbour; any other slab runs a general
 * kernel (uint8: a thread per active site; bits: a thread per 32-site word) in which every CTA waits and the
 * last CTA out posts.  pgg_get_variant_used() says which
 * (PGG_VARIANT_LEAN / PGG_VARIANT_V0); the environment variable PGG_SLAB_LEAN=0 forces the general kernel.
 * Errors: PGG_ERR_NULL, PGG_ERR_BAD_L, PGG_ERR_ALIGN, PGG_ERR_BAD_PARAM (rows, k_begin, r, K, span, epochs),
 * PGG_ERR_UNSUPPORTED (fmt, order_mode), PGG_ERR_CUDA.  n_phases == 0 is a no-op.
 * pgg_slab_alloc / pgg_slab_free: cudaMalloc'ed, zeroed memory of its own allocation (what an IPC handle
 * needs; torch tensors are carved out of larger blocks) -- both synchronise the device.
 * pgg_slab_ipc_export: 64-byte handle of such an allocation, to be sent to the neighbour processes;
 * pgg_slab_ipc_open: the neighbour's allocation mapped into this process (peer_device = the CUDA ordinal it
 * lives on, or -1 if unknown / the same device; PGG_ERR_UNSUPPORTED without a P2P path); pgg_slab_ipc_close. */
#define PGG_SLAB_MAX_MCS 4096u
#define PGG_SLAB_IPC_HANDLE_BYTES 64
uint64_t pgg_slab_bytes(int32_t fmt, uint32_t L, uint32_t n_rows);
/* Row granularity of the fast slab kernel: a slab whose row0 and n_rows are multiples of it runs LEAN's ring kernel
 * (L = 1024 .. 32768, a power of two: 4 R rows, R = LEAN's active rows per step for this layout), else 4.  Uses the
 * current CUDA device; 4 on any failure.                                                                          */
uint32_t pgg_slab_step_rows(int32_t fmt, uint32_t L);
int32_t pgg_slab_sweep(void* d_slab, int32_t fmt, uint32_t L, uint32_t row0, uint32_t n_rows, double r, double K,
                       uint64_t seed, int32_t order_mode, uint32_t t_begin, uint32_t k_begin, uint32_t n_phases,
                       void* d_up_halo, void* d_dn_halo, uint32_t* d_flags, uint32_t* d_up_flag, uint32_t* d_dn_flag,
                       uint32_t epoch0, uint64_t* d_deltas, void* stream);
/* The prisoner's dilemma (readings G1-G4 above, pgg_pd_sweep) on a row slab: pgg_slab_sweep with the payoffs
 * (R, S, T, P) in place of r -- same buffer, halo push, flags, kernels (LEAN's ring kernel or the general ones with the
 * game's table index), errors; the slabs together evolve bit for bit as pgg_pd_sweep evolves the unsharded lattice. */
int32_t pgg_pd_slab_sweep(void* d_slab, int32_t fmt, uint32_t L, uint32_t row0, uint32_t n_rows, double R, double S, double T,
                          double P, double K, uint64_t seed, int32_t order_mode, uint32_t t_begin, uint32_t k_begin,
                          uint32_t n_phases, void* d_up_halo, void* d_dn_halo, uint32_t* d_flags, uint32_t* d_up_flag,
                          uint32_t* d_dn_flag, uint32_t epoch0, uint64_t* d_deltas, void* stream);
int32_t pgg_slab_alloc(uint64_t bytes, void** d_out);
int32_t pgg_slab_free(void* d_ptr);
int32_t pgg_slab_ipc_export(void* d_ptr, uint8_t* h_handle64);
int32_t pgg_slab_ipc_open(const uint8_t* h_handle64, int32_t peer_device, void** d_out);
int32_t pgg_slab_ipc_close(void* d_ptr);

/* The 16 phase classes of MCS t, computed by the library's own
 * device kernel and copied back; h_out16: host array of 16 bytes.  Synchronises
 * `stream`.  For tests of step a1.  PGG_ORDER_DTILE has no classes:
 * PGG_ERR_UNSUPPORTED.                                                           */
int32_t pgg_phase_classes(uint64_t seed, uint32_t t, int32_t order_mode, uint8_t* h_out16,
                          void* stream);

/* Select the phase-kernel variant used by pgg_sweep / pgg_run_ensemble from now
 * on (process-wide; PGG_VARIANT_*).  Returns PGG_ERR_UNSUPPORTED if unknown.
 * pgg_get_variant_used() reports the variant the last sweep on this thread ran. */
int32_t pgg_set_variant(int32_t variant);
int32_t pgg_get_variant_used(void);

/* 1 if kernel variant `variant` can run lattices of layout fmt and size L, else 0. */
int32_t pgg_variant_supported(int32_t variant, int32_t fmt, uint32_t L);

/* ALU ceiling probe ("a Philox-only kernel's site-draws/s").  Enqueues ONE
 * launch of a kernel in which every thread of a full grid makes 2*iters STEP draws (the draw
 * of an elementary step, exactly as the phase kernels compute it: Philox4x32-10,
 * counter (site, t, (k<<8)|c, 3), words x0 and x1) and nothing else.  *h_n_draws (host, written
 * before return) = draws the launch makes; the caller times the launch with events on `stream`.
 * No lattice is touched.  Errors: PGG_ERR_NULL, PGG_ERR_BAD_PARAM (iters == 0), PGG_ERR_CUDA. */
int32_t pgg_probe_draw_rate(uint32_t iters, uint64_t seed, uint64_t* h_n_draws, void* stream);

/* Number of sites with at least one nearest neighbour of the other strategy: the sites for which
 * an elementary step needs its random draw (S9: for all others no draw can change
 * the state).  count / L^2 is the draw fraction of the state, the factor between the Philox-only
 * ceiling (pgg_probe_draw_rate) and the update rate it allows.  d_count: device uint64, overwritten.
 * Errors as pgg_density.                                                                      */
int32_t pgg_count_interface(const void* d_lat, int32_t fmt, uint32_t L, uint64_t* d_count, void* stream);

/* Number of kernels this library has launched in this process (monotone).       */
/* Temporaries (seeds, tables, class order, the PGG_VARIANT_PACKED working copy) come from a stream-ordered
 * memory pool the library owns, one per device; what a call frees stays in that pool for the next call
 * (at most the largest working set calls have had in flight at once).  This returns the unused part to the
 * driver for the current device; memory of calls still running on a stream is kept.  Errors: PGG_ERR_CUDA. */
int32_t pgg_trim_workspace(void);

uint64_t pgg_launch_count(void);

/* Text of the last error on the calling thread ("" if none).                    */
const char* pgg_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PGG_H_ */
