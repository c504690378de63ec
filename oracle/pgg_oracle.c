/*
 * pgg_oracle.c -- plain, slow, obviously-correct CPU oracle for the spatial
 * public goods game Monte Carlo sweep (Perc, arXiv:1704.08098).
 *
 * THIS FILE IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no
 * code, header, table or constant generator with the CUDA path under
 * paper_1704_08098_b200/csrc/ and neither side includes the other.
 *
 * Every function cites the passage of /root/reference/PAPER.md ("PAPER.md:<line>")
 * or the reading in SURVEY.md section 8(c) ("D1".."D8", "S1".."S20") it follows.
 * Floating point is IEEE double and appears only in the payoff/Fermi formulae and
 * in the 153-entry acceptance table; the lattice dynamics are integer-exact.
 *
 * Parity pins (tests/test_oracle_*.py): Philox known answers, closed-form
 * payoffs on hand-enumerated patches, the Fermi formula evaluated at 50 digits,
 * absorbing states, exact one-step law on all 2^16 states of the 4x4 torus,
 * visiting-order independence, composition.  Nothing here is "parity unpinned"
 * for the sublattice schedule; the random-sequential mode is pinned
 * statistically only (it is used for statistics only).
 *
 * Conventions ("Notation"):
 *   site (i,j), 0 <= i,j < L, row-major site = i*L + j, periodic in both axes.
 *   s in {0,1}: D = 0, C = 1 (d_x of Eq. 4).
 *   cross(z) = { z, z +- e_i, z +- e_j }  -- the von Neumann group centred on z,
 *   G = 5 members (Fig. 1).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_TAG_INIT 1u  /* D1: c3 tags */
#define ORC_TAG_ORDER 2u
#define ORC_TAG_STEP 3u
#define ORC_TAG_RS 4u
#define ORC_TAG_DTILE 5u /* T2: the paper's double-tiling schedule */

#define ORC_ORDER_IID 0  /* D5 */
#define ORC_ORDER_PERM 1
#define ORC_ORDER_DTILE 2 /* PAPER.md:75-93, readings T1-T4 */

/* ------------------------------------------------------------------------- */
/* D1. Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  The paper only says */
/* "random"; north_star fixes Philox4x32, S5 fixes 10 rounds.    */
/* ------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; /* key bump after each round */
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static void seed_key(uint64_t seed, uint32_t key[2])
{
    key[0] = (uint32_t)(seed & 0xFFFFFFFFu); /* D1: key = (seed lo, seed hi) */
    key[1] = (uint32_t)(seed >> 32);
}

/* ------------------------------------------------------------------------- */
/* Lattice access with periodic boundaries.                     */
/* ------------------------------------------------------------------------- */
static inline int wrap(int a, int L)
{
    a %= L;
    return a < 0 ? a + L : a;
}

static inline int s_at(const uint8_t *lat, int L, int i, int j)
{
    return lat[(size_t)wrap(i, L) * (size_t)L + (size_t)wrap(j, L)];
}

/* N(z): number of cooperators N_C in the group centred on z=(i,j) -- the     */
/* centre and its four nearest neighbours (S10: x counts itself). */
int orc_group_count(const uint8_t *lat, int L, int i, int j)
{
    return s_at(lat, L, i, j) + s_at(lat, L, i - 1, j) + s_at(lat, L, i + 1, j) +
           s_at(lat, L, i, j - 1) + s_at(lat, L, i, j + 1);
}

/* D2, literal form.  Player x=(i,j) is a member of the G=5 groups centred on  */
/* the sites of cross(x).  From each it earns                 */
/*   Pi_C^g = r*c*N_C/G - c   or   Pi_D^g = r*c*N_C/G,   c = 1   (Eqs. 1-2,   */
/* PAPER.md:47-50), and its total payoff is the sum over the five groups       */
/* (PAPER.md:54,56).  S10: the cost c is paid once per group.                  */
double orc_payoff_literal(const uint8_t *lat, int L, int i, int j, double r)
{
    static const int di[5] = {0, -1, 1, 0, 0};
    static const int dj[5] = {0, 0, 0, -1, 1};
    const double G = 5.0, c = 1.0;
    int sx = s_at(lat, L, i, j);
    double total = 0.0;
    for (int g = 0; g < 5; ++g) {
        int NC = orc_group_count(lat, L, i + di[g], j + dj[g]);
        double pi_g = r * c * (double)NC / G;
        if (sx == 1)
            pi_g -= c;
        total += pi_g;
    }
    return total;
}

/* Integer payoff kernel A_x = sum over the five groups of N(z)  (D2).  With   */
/* c=1, G=5:  Pi_x = (r/5)*A_x - 5*s_x.                                        */
int orc_A(const uint8_t *lat, int L, int i, int j)
{
    return orc_group_count(lat, L, i, j) + orc_group_count(lat, L, i - 1, j) +
           orc_group_count(lat, L, i + 1, j) + orc_group_count(lat, L, i, j - 1) +
           orc_group_count(lat, L, i, j + 1);
}

/* Eq. (3):  W(s_y -> s_x) = 1 / (1 + exp[(Pi_x - Pi_y)/K]).      */
/* S12: this is the probability that x adopts the strategy of y.               */
double orc_fermi(double Pi_x, double Pi_y, double K)
{
    return 1.0 / (1.0 + exp((Pi_x - Pi_y) / K));
}

/* ------------------------------------------------------------------------- */
/* D3. Acceptance table.  Pi_x - Pi_y depends only on dA = A_x - A_y in        */
/* [-25,25] and ds = s_x - s_y in {-1,0,1} (north_star); the uniform deviate   */
/* is a uint32 u and x adopts s_y iff u < T[(ds+1)*51 + (dA+25)].             */
/* Operation order fixed by D3; S7: clamp when W*2^32 does not fit.            */
/* ------------------------------------------------------------------------- */
int orc_table_index(int dA, int ds)
{
    return (ds + 1) * 51 + (dA + 25);
}

void orc_accept_table(double r, double K, uint32_t out153[153])
{
    for (int ds = -1; ds <= 1; ++ds) {
        for (int dA = -25; dA <= 25; ++dA) {
            double delta = (r * (double)dA) / 5.0 - 5.0 * (double)ds; /* Pi_x - Pi_y */
            double z = delta / K;
            double W = 1.0 / (1.0 + exp(z));
            double v = W * 4294967296.0;
            uint32_t T;
            if (v >= 4294967295.0)
                T = 0xFFFFFFFFu;
            else
                T = (uint32_t)floor(v);
            out153[orc_table_index(dA, ds)] = T;
        }
    }
}

/* ------------------------------------------------------------------------- */
/* D4. Initial condition: each site C or D with probability rho0 / 1-rho0      */
/* ("with equal probability" => rho0 = 0.5).                      */
/* ------------------------------------------------------------------------- */
void orc_init(uint8_t *lat, int L, double rho0, uint64_t seed)
{
    uint32_t key[2];
    seed_key(seed, key);
    uint64_t thr = (uint64_t)floor(rho0 * 4294967296.0);
    size_t n = (size_t)L * (size_t)L;
    for (size_t site = 0; site < n; ++site) {
        uint32_t ctr[4] = {(uint32_t)site, 0u, 0u, ORC_TAG_INIT};
        uint32_t x[4];
        orc_philox4x32_10(ctr, key, x);
        lat[site] = ((uint64_t)x[0] < thr) ? 1 : 0;
    }
}

/* Eq. (4) numerator: sum_x d_x.                                  */
uint64_t orc_count(const uint8_t *lat, int L)
{
    uint64_t n = 0;
    size_t sz = (size_t)L * (size_t)L;
    for (size_t a = 0; a < sz; ++a)
        n += lat[a];
    return n;
}

/* ------------------------------------------------------------------------- */
/* D5. The 16 sublattice classes visited in MCS t.  class(i,j) =               */
/* 4*(i mod 4) + (j mod 4)  (north_star: "16 sublattices by (i mod 4, j mod    */
/* 4)", visited "in a Philox-drawn order").  S2: IID = each of the 16 phases   */
/* draws its class uniformly (default); PERM = a permutation of the classes.   */
/* ------------------------------------------------------------------------- */
void orc_phase_classes(uint64_t seed, uint32_t t, int order_mode, uint8_t out16[16])
{
    uint32_t key[2];
    seed_key(seed, key);
    uint32_t w[16];
    for (uint32_t q = 0; q < 4; ++q) {
        uint32_t ctr[4] = {t, 0u, q, ORC_TAG_ORDER};
        orc_philox4x32_10(ctr, key, &w[4 * q]);
    }
    if (order_mode == ORC_ORDER_IID) {
        for (int k = 0; k < 16; ++k)
            out16[k] = (uint8_t)(w[k] >> 28);
    } else {
        /* classes sorted ascending by (w[c], c); phase k takes the k-th */
        int used[16] = {0};
        for (int k = 0; k < 16; ++k) {
            int best = -1;
            for (int c = 0; c < 16; ++c) {
                if (used[c])
                    continue;
                if (best < 0 || w[c] < w[best]) /* ties: lower c first (scan order) */
                    best = c;
            }
            used[best] = 1;
            out16[k] = (uint8_t)best;
        }
    }
}

/* ------------------------------------------------------------------------- */
/* One elementary step for a given focal site, direction and     */
/* uniform deviate.  Returns the strategy of x after the step; does not write. */
/* dir: 0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1)  (D6).                         */
/* ------------------------------------------------------------------------- */
int orc_step_given_draw(const uint8_t *lat, int L, const uint32_t table[153], int i, int j,
                        int dir, uint32_t u)
{
    static const int di[4] = {-1, 1, 0, 0};
    static const int dj[4] = {0, 0, -1, 1};
    int yi = i + di[dir], yj = j + dj[dir];
    int sx = s_at(lat, L, i, j);
    int sy = s_at(lat, L, yi, yj);
    if (sx == sy)
        return sx; /* S9: copying one's own strategy changes nothing */
    int Ax = orc_A(lat, L, i, j);   /* x plays in all its G groups */
    int Ay = orc_A(lat, L, yi, yj); /* so does y (S11)                           */
    uint32_t T = table[orc_table_index(Ax - Ay, sx - sy)];
    return (u < T) ? sy : sx; /* strict: accept iff u < T (D3) */
}

/* Threshold T such that x=(i,j) adopts the strategy of its neighbour in       */
/* direction dir iff u < T; 0 when s_y == s_x.  (The one-step law is           */
/* P(flip) = 1/4 * sum_dir T/2^32; pinned by brute force on the 4x4 torus.)    */
uint32_t orc_flip_threshold(const uint8_t *lat, int L, const uint32_t table[153], int i, int j,
                            int dir)
{
    static const int di[4] = {-1, 1, 0, 0};
    static const int dj[4] = {0, 0, -1, 1};
    int yi = i + di[dir], yj = j + dj[dir];
    int sx = s_at(lat, L, i, j);
    int sy = s_at(lat, L, yi, yj);
    if (sx == sy)
        return 0u;
    return table[orc_table_index(orc_A(lat, L, i, j) - orc_A(lat, L, yi, yj), sx - sy)];
}

/* Batch form for the 4x4 brute-force pin: for each of n_states lattices (L*L  */
/* bytes each), every site and every direction, the threshold above.           */
void orc_flip_thresholds_batch(const uint8_t *lats, int n_states, int L, const uint32_t table[153],
                               uint32_t *out /* [n_states][L*L][4] */)
{
    size_t n = (size_t)L * (size_t)L;
    for (int a = 0; a < n_states; ++a)
        for (int i = 0; i < L; ++i)
            for (int j = 0; j < L; ++j)
                for (int dir = 0; dir < 4; ++dir)
                    out[((size_t)a * n + (size_t)i * L + j) * 4 + dir] =
                        orc_flip_threshold(lats + (size_t)a * n, L, table, i, j, dir);
}

/* The STEP draw of site `site` in phase k (class c) of MCS t  (D6, S3).       */
void orc_step_draw(uint64_t seed, uint32_t site, uint32_t t, uint32_t k, uint32_t c, int *dir,
                   uint32_t *u)
{
    uint32_t key[2];
    seed_key(seed, key);
    uint32_t ctr[4] = {site, t, (k << 8) | c, ORC_TAG_STEP};
    uint32_t x[4];
    orc_philox4x32_10(ctr, key, x);
    *dir = (int)(x[0] >> 30);
    *u = x[1];
}

/* ------------------------------------------------------------------------- */
/* D6. Phase k of MCS t, class c = 4*ci + cj: every site with i%4==ci,         */
/* j%4==cj performs one elementary step, in place.  Race-free by S1: a step at */
/* x reads only sites within Manhattan distance 3 of x and writes only x, and  */
/* two sites of one class are >= 4 apart (needs L % 4 == 0).  visit: 0 raster, */
/* 1 reverse raster, 2 = the order given in perm[] (indices into the raster    */
/* list of the class) -- the result must not depend on it (pin P6).            */
/* Returns the signed change of the cooperator count.                          */
/* n_threads > 1 splits the rows of the class over OpenMP threads (same        */
/* result, by S1); used only to bound the wall time of large parity runs.      */
/* ------------------------------------------------------------------------- */
int64_t orc_phase(uint8_t *lat, int L, const uint32_t table[153], uint64_t seed, uint32_t t,
                  uint32_t k, uint32_t c, int visit, const uint32_t *perm, int n_threads)
{
    int ci = (int)(c >> 2), cj = (int)(c & 3u);
    int m = L / 4; /* class sites per row / column */
    int64_t delta = 0;
    if (n_threads <= 1 || visit != 0) {
        size_t n_cls = (size_t)m * (size_t)m;
        for (size_t a = 0; a < n_cls; ++a) {
            size_t b = a;
            if (visit == 1)
                b = n_cls - 1 - a;
            else if (visit == 2)
                b = perm[a];
            int i = 4 * (int)(b / (size_t)m) + ci;
            int j = 4 * (int)(b % (size_t)m) + cj;
            uint32_t site = (uint32_t)((size_t)i * (size_t)L + (size_t)j);
            int dir;
            uint32_t u;
            orc_step_draw(seed, site, t, k, c, &dir, &u);
            int old = lat[site];
            int neu = orc_step_given_draw(lat, L, table, i, j, dir, u);
            lat[site] = (uint8_t)neu;
            delta += neu - old;
        }
    } else {
#ifdef _OPENMP
#pragma omp parallel for num_threads(n_threads) reduction(+ : delta) schedule(static)
#endif
        for (int bi = 0; bi < m; ++bi) {
            int i = 4 * bi + ci;
            for (int bj = 0; bj < m; ++bj) {
                int j = 4 * bj + cj;
                uint32_t site = (uint32_t)((size_t)i * (size_t)L + (size_t)j);
                int dir;
                uint32_t u;
                orc_step_draw(seed, site, t, k, c, &dir, &u);
                int old = lat[site];
                int neu = orc_step_given_draw(lat, L, table, i, j, dir, u);
                lat[site] = (uint8_t)neu;
                delta += neu - old;
            }
        }
    }
    return delta;
}

/* ------------------------------------------------------------------------- */
/* The paper's own parallel schedule: double tiling decomposition              */
/* (Fig. 2, Fig. 3).  The lattice is cut into 4x4 domains      */
/* ("domain size S to be 4x4"); domain (I,J) = (i>>2, j>>2) has    */
/* type 2*(I&1) + (J&1) in {0,1,2,3} -- the paper's types 1,2,3,4, laid out    */
/* "linearly in sequences of 2 (1,2,1,2,... or 3,4,3,4,...)", so */
/* L % 8 == 0.  A full MCS is four parts, the types "updated  */
/* in turn" 1,2,3,4; in a part every domain of that type is      */
/* updated by "independent parallel random sequential updating". */
/* Readings where the paper is silent (S15, T1-T4):       */
/*  T1 picks per domain per part = 16 = the domain's sites, so that one MCS is */
/*     4 parts x L^2/64 domains x 16 = L^2 elementary steps;     */
/*  T2 pick p of domain d = I*(L/4)+J in MCS t draws (x0,x1,x2,.) =            */
/*     Philox(ctr = (d, t, p, DTILE)); focal site = domain row x0>>30, domain  */
/*     column (x0>>28)&3; neighbour direction = x2>>30 (as D6); u = x1;        */
/*  T3 domain origins are fixed (no shift between MCS);                        */
/*  T4 the picks of one domain are sequential: pick p sees picks 0..p-1.       */
/* Race freedom: a step reads within Manhattan distance 3 of x (S1) and writes */
/* x; two domains of one type are separated by a 4-site gap in each axis, so   */
/* no read of one reaches into the other ("three lines outward").  */
/* ------------------------------------------------------------------------- */
int orc_dtile_type(int I, int J)
{
    return 2 * (I & 1) + (J & 1);
}

void orc_dtile_draw(uint64_t seed, uint32_t d, uint32_t t, uint32_t p, int *a, int *b, int *dir,
                    uint32_t *u)
{
    uint32_t key[2];
    seed_key(seed, key);
    uint32_t ctr[4] = {d, t, p, ORC_TAG_DTILE};
    uint32_t x[4];
    orc_philox4x32_10(ctr, key, x);
    *a = (int)(x[0] >> 30);
    *b = (int)((x[0] >> 28) & 3u);
    *dir = (int)(x[2] >> 30);
    *u = x[1];
}

/* The 16 sequential elementary steps of domain (I,J) in MCS t (T1, T4).       */
static int64_t dtile_domain(uint8_t *lat, int L, const uint32_t table[153], uint64_t seed,
                            uint32_t t, int I, int J)
{
    int64_t delta = 0;
    uint32_t d = (uint32_t)(I * (L / 4) + J);
    for (uint32_t p = 0; p < 16; ++p) {
        int a, b, dir;
        uint32_t u;
        orc_dtile_draw(seed, d, t, p, &a, &b, &dir, &u);
        int i = 4 * I + a, j = 4 * J + b;
        size_t site = (size_t)i * (size_t)L + (size_t)j;
        int old = lat[site];
        int neu = orc_step_given_draw(lat, L, table, i, j, dir, u);
        lat[site] = (uint8_t)neu;
        delta += neu - old;
    }
    return delta;
}

/* Part q of MCS t: every domain of type q.  visit: 0 raster over the domains, */
/* 1 reverse raster -- the result must not depend on it.  n_threads > 1 splits */
/* the domain rows over OpenMP threads (same result, by the race freedom       */
/* above).  Returns the signed change of the cooperator count.                 */
int64_t orc_dtile_part(uint8_t *lat, int L, const uint32_t table[153], uint64_t seed, uint32_t t,
                       int q, int visit, int n_threads)
{
    int M = L / 4;
    int64_t delta = 0;
    if (n_threads <= 1 || visit != 0) {
        for (int n = 0; n < M * M; ++n) {
            int m = visit == 1 ? M * M - 1 - n : n;
            int I = m / M, J = m % M;
            if (orc_dtile_type(I, J) == q)
                delta += dtile_domain(lat, L, table, seed, t, I, J);
        }
    } else {
#ifdef _OPENMP
#pragma omp parallel for num_threads(n_threads) reduction(+ : delta) schedule(static)
#endif
        for (int I = 0; I < M; ++I)
            for (int J = 0; J < M; ++J)
                if (orc_dtile_type(I, J) == q)
                    delta += dtile_domain(lat, L, table, seed, t, I, J);
    }
    return delta;
}

/* ------------------------------------------------------------------------- */
/* D6+D7. n_mcs full Monte Carlo steps t = t_begin .. t_begin+n_mcs-1, each 16 */
/* phases (1 MCS = L^2 elementary steps: 16 phases x L^2/16), or  */
/* with order_mode == ORC_ORDER_DTILE the four parts of the paper's schedule.  */
/* counts[m] = number of cooperators after MCS t_begin+m completes (may be     */
/* NULL).  If snap_every > 0, the lattice is copied to snaps after every MCS   */
/* whose 1-based index within this call is a multiple of snap_every.           */
/* Returns 0, or -1 on bad arguments.                                          */
/* ------------------------------------------------------------------------- */
int orc_sweep(uint8_t *lat, int L, double r, double K, uint64_t seed, int order_mode,
              uint32_t t_begin, uint32_t n_mcs, uint64_t *counts, uint32_t snap_every,
              uint8_t *snaps, int n_threads)
{
    if (L < 4 || L % 4 != 0 || !(K > 0.0))
        return -1;
    if (order_mode == ORC_ORDER_DTILE && L % 8 != 0)
        return -1;
    uint32_t table[153];
    orc_accept_table(r, K, table);
    size_t n = (size_t)L * (size_t)L;
    int64_t count = (int64_t)orc_count(lat, L);
    size_t n_snap = 0;
    for (uint32_t m = 0; m < n_mcs; ++m) {
        uint32_t t = t_begin + m;
        if (order_mode == ORC_ORDER_DTILE) {
            for (int q = 0; q < 4; ++q) /* types 1,2,3,4 in turn */
                count += orc_dtile_part(lat, L, table, seed, t, q, 0, n_threads);
        } else {
            uint8_t cls[16];
            orc_phase_classes(seed, t, order_mode, cls);
            for (uint32_t k = 0; k < 16; ++k)
                count += orc_phase(lat, L, table, seed, t, k, cls[k], 0, NULL, n_threads);
        }
        if (counts)
            counts[m] = (uint64_t)count;
        if (snap_every > 0 && (m + 1) % snap_every == 0) {
            memcpy(snaps + n_snap * n, lat, n);
            ++n_snap;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* D8. Classic random sequential update: L^2 times per MCS    */
/* pick x uniformly, pick y among its four neighbours, adopt with W.  Used for */
/* statistical comparison only.  g is the global elementary-step counter.      */
/* ------------------------------------------------------------------------- */
int orc_rs_sweep(uint8_t *lat, int L, double r, double K, uint64_t seed, uint64_t g_begin,
                 uint32_t n_mcs, uint64_t *counts)
{
    if (L < 4 || !(K > 0.0))
        return -1;
    uint32_t table[153];
    orc_accept_table(r, K, table);
    uint32_t key[2];
    seed_key(seed, key);
    uint64_t n = (uint64_t)L * (uint64_t)L;
    int64_t count = (int64_t)orc_count(lat, L);
    uint64_t g = g_begin;
    for (uint32_t m = 0; m < n_mcs; ++m) {
        for (uint64_t a = 0; a < n; ++a, ++g) {
            uint32_t ctr[4] = {(uint32_t)(g & 0xFFFFFFFFu), (uint32_t)(g >> 32), 0u, ORC_TAG_RS};
            uint32_t x[4];
            orc_philox4x32_10(ctr, key, x);
            uint64_t site = ((uint64_t)x[0] * n) >> 32;
            int i = (int)(site / (uint64_t)L), j = (int)(site % (uint64_t)L);
            int dir = (int)(x[2] >> 30);
            uint32_t u = x[3];
            int old = lat[site];
            int neu = orc_step_given_draw(lat, L, table, i, j, dir, u);
            lat[site] = (uint8_t)neu;
            count += neu - old;
        }
        if (counts)
            counts[m] = (uint64_t)count;
    }
    return 0;
}

/* Canonical bit-packed I/O layout: site (i,j) is bit */
/* (j & 31) of the little-endian uint32 word i*(L/32) + (j >> 5); L % 32 == 0. */
void orc_pack_bits(const uint8_t *lat, int L, uint32_t *words)
{
    size_t wpr = (size_t)L / 32;
    memset(words, 0, (size_t)L * wpr * sizeof(uint32_t));
    for (int i = 0; i < L; ++i)
        for (int j = 0; j < L; ++j)
            if (lat[(size_t)i * L + j])
                words[(size_t)i * wpr + (size_t)(j >> 5)] |= (1u << (j & 31));
}

void orc_unpack_bits(const uint32_t *words, int L, uint8_t *lat)
{
    size_t wpr = (size_t)L / 32;
    for (int i = 0; i < L; ++i)
        for (int j = 0; j < L; ++j)
            lat[(size_t)i * L + j] =
                (uint8_t)((words[(size_t)i * wpr + (size_t)(j >> 5)] >> (j & 31)) & 1u);
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
