/*
 * pd_oracle.c -- plain CPU oracle for the spatial PRISONER'S DILEMMA on the square lattice, the
 * "other evolutionary game" the paper names as the first adaptation of its scheme (PAPER.md:131,
 * section VI): "the prisoner's dilemma game is played in a pairwise manner, not in groups.  As a
 * consequence, the memory needed to update strategies within a given domain is one line outward
 * less in each direction".
 *
 * THIS FILE IS TEST INFRASTRUCTURE (as pgg_oracle.c): only tests/ and __graft_entry__.smoke() may
 * load it; it shares nothing with the CUDA path.  It reuses pgg_oracle.c's public Philox, phase
 * class and STEP draw functions (the schedule and the random numbers are those of the public goods
 * game: D1, D5, D6); everything the game itself defines is written out here.
 *
 * The paper gives no payoff matrix.  Readings (G1-G4):
 *  G1 payoff: x plays one two-player game with each of its four nearest neighbours (no game with
 *     itself).  A pair earns: C against C -> R, C against D -> S, D against C -> T, D against D -> P
 *     (the usual names; the weak dilemma of the literature the paper cites is R = 1, S = P = 0,
 *     T = b).  Pi_x = sum over the four neighbours y of payoff(s_x, s_y).
 *  G2 update: the elementary step, the Fermi rule Eq. (3) and the 16-sublattice
 *     Philox schedule are unchanged; only Pi changes.
 *  G3 table: with n_z = number of cooperators among the four neighbours of z,
 *     Pi_z = s_z ? R n_z + S (4 - n_z) : T n_z + P (4 - n_z).  A step matters only if s_y = 1 - s_x,
 *     so the acceptance threshold depends on (s_x, n_x, n_y): 50 entries at s_x*25 + n_x*5 + n_y,
 *     in IEEE double in exactly this order:  z = (Pi_x - Pi_y)/K;  W = 1/(1 + exp(z));
 *     v = W * 2^32;  T = v >= 4294967295 ? 0xFFFFFFFF : floor(v).  Accept iff u < T (strict).
 *  G4 halo: a step at x reads x, y and their neighbours: Manhattan distance <= 2 from x
 *     ("one line outward less"); sites of one class are >= 4 apart, so the schedule
 *     stays race-free.
 *
 * Pins (tests/test_oracle_pd.py): closed-form payoffs (all-C 4R, all-D 4P, lone defector 4T among
 * neighbours earning 3R + S, lone cooperator 4S, checkerboard), the pairwise sum against the count
 * form, the table against a 60-digit evaluation of Eq. (3), the exact one-step law on all 2^16
 * states of the 4x4 torus with payoffs from numpy rolls, the radius-2 read stencil, strictness of
 * u < T in every direction, absorbing states, order independence, composition.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* from pgg_oracle.c (same shared library) */
void orc_phase_classes(uint64_t seed, uint32_t t, int order_mode, uint8_t out16[16]);
void orc_step_draw(uint64_t seed, uint32_t site, uint32_t t, uint32_t k, uint32_t c, int *dir, uint32_t *u);
uint64_t orc_count(const uint8_t *lat, int L);

static inline int pd_wrap(int a, int L)
{
    a %= L;
    return a < 0 ? a + L : a;
}

static inline int pd_s(const uint8_t *lat, int L, int i, int j)
{
    return lat[(size_t)pd_wrap(i, L) * (size_t)L + (size_t)pd_wrap(j, L)];
}

/* G1, literal: the sum of the four pair games of x = (i,j).  pay[2][2] = {{P, T}, {S, R}} indexed  */
/* [s_x][s_y]: what x earns against y.                                                             */
double orc_pd_payoff_literal(const uint8_t *lat, int L, int i, int j, double R, double S, double T, double P)
{
    static const int di[4] = {-1, 1, 0, 0};
    static const int dj[4] = {0, 0, -1, 1};
    int sx = pd_s(lat, L, i, j);
    double total = 0.0;
    for (int q = 0; q < 4; ++q) {
        int sy = pd_s(lat, L, i + di[q], j + dj[q]);
        if (sx == 1)
            total += sy == 1 ? R : S;
        else
            total += sy == 1 ? T : P;
    }
    return total;
}

/* n_z: cooperators among the four nearest neighbours of z (z itself not counted). */
int orc_pd_nc(const uint8_t *lat, int L, int i, int j)
{
    return pd_s(lat, L, i - 1, j) + pd_s(lat, L, i + 1, j) + pd_s(lat, L, i, j - 1) + pd_s(lat, L, i, j + 1);
}

/* G3, count form of the payoff. */
double orc_pd_payoff(int s, int n, double R, double S, double T, double P)
{
    return s == 1 ? R * (double)n + S * (double)(4 - n) : T * (double)n + P * (double)(4 - n);
}

int orc_pd_table_index(int sx, int nx, int ny)
{
    return sx * 25 + nx * 5 + ny;
}

/* G3: the 50 thresholds.  volatile keeps the stated operation order under any optimiser. */
void orc_pd_accept_table(double R, double S, double T, double P, double K, uint32_t out[50])
{
    for (int sx = 0; sx <= 1; ++sx)
        for (int nx = 0; nx <= 4; ++nx)
            for (int ny = 0; ny <= 4; ++ny) {
                volatile double Px = orc_pd_payoff(sx, nx, R, S, T, P);
                volatile double Py = orc_pd_payoff(1 - sx, ny, R, S, T, P);
                volatile double z = (Px - Py) / K;
                volatile double W = 1.0 / (1.0 + exp(z));
                double v = W * 4294967296.0;
                out[orc_pd_table_index(sx, nx, ny)] = v >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)floor(v);
            }
}

/* Threshold below which x = (i,j) adopts the strategy of its neighbour in direction dir            */
/* (0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1), D6); 0 when s_y == s_x.                                 */
uint32_t orc_pd_flip_threshold(const uint8_t *lat, int L, const uint32_t table[50], int i, int j, int dir)
{
    static const int di[4] = {-1, 1, 0, 0};
    static const int dj[4] = {0, 0, -1, 1};
    int yi = i + di[dir], yj = j + dj[dir];
    int sx = pd_s(lat, L, i, j), sy = pd_s(lat, L, yi, yj);
    if (sx == sy)
        return 0u;
    return table[orc_pd_table_index(sx, orc_pd_nc(lat, L, i, j), orc_pd_nc(lat, L, yi, yj))];
}

/* One elementary step for a given focal site, direction and deviate; returns the     */
/* strategy of x after the step, does not write.                                                    */
int orc_pd_step_given_draw(const uint8_t *lat, int L, const uint32_t table[50], int i, int j, int dir, uint32_t u)
{
    int sx = pd_s(lat, L, i, j);
    uint32_t T = orc_pd_flip_threshold(lat, L, table, i, j, dir);
    return (u < T) ? 1 - sx : sx; /* strict; T = 0 when s_y == s_x */
}

/* Phase k of MCS t, class c (D6 with the pair-game payoffs).  visit: 0 raster, 1 reverse raster.   */
int64_t orc_pd_phase(uint8_t *lat, int L, const uint32_t table[50], uint64_t seed, uint32_t t, uint32_t k,
                     uint32_t c, int visit)
{
    int ci = (int)(c >> 2), cj = (int)(c & 3u), m = L / 4;
    size_t n_cls = (size_t)m * (size_t)m;
    int64_t delta = 0;
    for (size_t a = 0; a < n_cls; ++a) {
        size_t b = visit == 1 ? n_cls - 1 - a : a;
        int i = 4 * (int)(b / (size_t)m) + ci, j = 4 * (int)(b % (size_t)m) + cj;
        uint32_t site = (uint32_t)((size_t)i * (size_t)L + (size_t)j);
        int dir;
        uint32_t u;
        orc_step_draw(seed, site, t, k, c, &dir, &u);
        int old = lat[site];
        int neu = orc_pd_step_given_draw(lat, L, table, i, j, dir, u);
        lat[site] = (uint8_t)neu;
        delta += neu - old;
    }
    return delta;
}

/* n_mcs full MCS (16 phases each, classes by D5); counts[m] = cooperators after MCS t_begin + m.   */
int orc_pd_sweep(uint8_t *lat, int L, double R, double S, double T, double P, double K, uint64_t seed,
                 int order_mode, uint32_t t_begin, uint32_t n_mcs, uint64_t *counts)
{
    if (L < 4 || L % 4 != 0 || !(K > 0.0) || (order_mode != 0 && order_mode != 1))
        return -1;
    uint32_t table[50];
    orc_pd_accept_table(R, S, T, P, K, table);
    int64_t count = (int64_t)orc_count(lat, L);
    for (uint32_t m = 0; m < n_mcs; ++m) {
        uint8_t cls[16];
        orc_phase_classes(seed, t_begin + m, order_mode, cls);
        for (uint32_t k = 0; k < 16; ++k)
            count += orc_pd_phase(lat, L, table, seed, t_begin + m, k, cls[k], 0);
        if (counts)
            counts[m] = (uint64_t)count;
    }
    return 0;
}
