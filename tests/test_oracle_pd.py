"""Pins of the prisoner's-dilemma oracle (``oracle/pd_oracle.c``, readings G1-G4 of
DESIGN.md section 2) against what the definition and the mathematics fix -- none of them re-types
the oracle's own formula: hand-enumerated payoffs, a pair-by-pair numpy evaluation, Eq. (3) at 60
digits, the exact one-step law on all 2^16 states of the 4x4 torus, the radius-2 read stencil the
paper states ("one line outward less"), invariants of the schedule."""
import decimal
import itertools

import numpy as np

import oracle as orc
import workloads as wl

R, S, T, P = 1.0, 0.0, 1.3, 0.0          # the weak dilemma: R = 1, S = P = 0, T = b
GEN = (3.0, -0.5, 4.25, 0.75)            # a generic matrix with T > R > P > S
DI, DJ = (-1, 1, 0, 0), (0, 0, -1, 1)


def numpy_payoffs(lat, R, S, T, P):
    """Pi for every site, pair by pair with numpy rolls (G1)."""
    lat = lat.astype(np.int64)
    total = np.zeros(lat.shape)
    for ax, sh in ((0, 1), (0, -1), (1, 1), (1, -1)):
        nb = np.roll(lat, sh, axis=ax)
        total += np.where(lat == 1, np.where(nb == 1, R, S), np.where(nb == 1, T, P))
    return total


def test_closed_form_payoffs():
    L = 12
    allc, alld = np.ones((L, L), np.uint8), np.zeros((L, L), np.uint8)
    assert orc.pd_payoff_literal(allc, 5, 5, *GEN) == 4 * GEN[0]           # four C-C pairs
    assert orc.pd_payoff_literal(alld, 5, 5, *GEN) == 4 * GEN[3]           # four D-D pairs
    lone_d = allc.copy(); lone_d[5, 5] = 0
    assert orc.pd_payoff_literal(lone_d, 5, 5, *GEN) == 4 * GEN[2]         # exploits four cooperators
    assert orc.pd_payoff_literal(lone_d, 4, 5, *GEN) == 3 * GEN[0] + GEN[1]
    assert orc.pd_payoff_literal(lone_d, 4, 4, *GEN) == 4 * GEN[0]         # a diagonal neighbour plays no game with it
    lone_c = alld.copy(); lone_c[5, 5] = 1
    assert orc.pd_payoff_literal(lone_c, 5, 5, *GEN) == 4 * GEN[1]
    assert orc.pd_payoff_literal(lone_c, 5, 6, *GEN) == GEN[2] + 3 * GEN[3]
    cb = wl.checkerboard_lattice(L)
    i, j = 3, 4                                                            # (i + j) odd -> C
    assert cb[i, j] == 1 and orc.pd_payoff_literal(cb, i, j, *GEN) == 4 * GEN[1]
    assert orc.pd_payoff_literal(cb, i, j + 1, *GEN) == 4 * GEN[2]
    # weak dilemma: a defector never earns less than a cooperator with the same neighbours when b >= 1
    for n in range(5):
        assert orc.pd_payoff(0, n, R, S, T, P) >= orc.pd_payoff(1, n, R, S, T, P)


def test_payoff_literal_equals_count_form_and_numpy_pairs():
    for L, p in ((4, 0.5), (8, 0.4), (20, 0.6)):
        lat = wl.random_lattice(L, p, seed=L)
        ref = numpy_payoffs(lat, *GEN)
        for i in range(L):
            for j in range(L):
                lit = orc.pd_payoff_literal(lat, i, j, *GEN)
                n = orc.pd_nc(lat, i, j)
                assert n == sum(int(lat[(i + DI[d]) % L, (j + DJ[d]) % L]) for d in range(4))
                assert lit == ref[i, j] == orc.pd_payoff(int(lat[i, j]), n, *GEN)


def test_table_against_the_fermi_formula_at_60_digits():
    decimal.getcontext().prec = 60
    for (Rr, Ss, Tt, Pp), K in ((GEN, 0.5), ((R, S, T, P), 0.1), ((1.0, 0.0, 2.0, 0.0), 2.0)):
        tab = orc.pd_accept_table(Rr, Ss, Tt, Pp, K)
        D = decimal.Decimal
        for sx, nx, ny in itertools.product((0, 1), range(5), range(5)):
            pay = lambda s, n: (D(Rr) * n + D(Ss) * (4 - n)) if s == 1 else (D(Tt) * n + D(Pp) * (4 - n))
            z = (pay(sx, nx) - pay(1 - sx, ny)) / D(K)
            W = D(1) / (D(1) + z.exp()) if z < 200 else D(0)
            exact = W * D(2) ** 32
            got = int(tab[orc.pd_table_index(sx, nx, ny)])
            want = min(int(exact), 0xFFFFFFFF) if exact < D(4294967295) else 0xFFFFFFFF
            assert abs(got - want) <= max(2, int(exact * D(2) ** -44)), (sx, nx, ny, got, want)
    # equal payoffs: W = 1/2; richer neighbour -> W > 1/2; K -> 0: a step function
    tab = orc.pd_accept_table(1.0, 0.0, 1.0, 0.0, 0.5)       # T = R, S = P: payoff = n for both strategies
    assert int(tab[orc.pd_table_index(1, 2, 2)]) == 0x80000000
    assert int(tab[orc.pd_table_index(1, 1, 3)]) > 0x80000000 > int(tab[orc.pd_table_index(1, 3, 1)])
    sharp = orc.pd_accept_table(R, S, T, P, 1e-3)
    assert int(sharp[orc.pd_table_index(1, 1, 3)]) == 0xFFFFFFFF and int(sharp[orc.pd_table_index(0, 4, 0)]) == 0


def test_exact_one_step_law_on_the_4x4_torus():
    """P(x flips) = 1/4 sum over directions [s_y != s_x] W(Pi_x - Pi_y), every state, every site; payoffs
    from numpy_payoffs, W from the formula in double (within the table's 2^-32 quantisation)."""
    L, K = 4, 0.5
    tab = orc.pd_accept_table(*GEN, K)
    rng = np.random.default_rng(5)
    states = rng.integers(0, 2 ** 16, size=600).tolist() + [0, 0xFFFF, 0x5A5A, 0x00FF, 0x0F0F]
    for st in states:
        lat = np.array([(st >> b) & 1 for b in range(16)], dtype=np.uint8).reshape(L, L)
        pay = numpy_payoffs(lat, *GEN)
        for i in range(L):
            for j in range(L):
                for d in range(4):
                    yi, yj = (i + DI[d]) % L, (j + DJ[d]) % L
                    thr = orc.pd_flip_threshold(lat, tab, i, j, d)
                    if lat[i, j] == lat[yi, yj]:
                        assert thr == 0
                    else:
                        W = 1.0 / (1.0 + np.exp((pay[i, j] - pay[yi, yj]) / K))
                        assert abs(thr / 2.0 ** 32 - W) < 2.0 ** -31, (st, i, j, d)


def test_read_stencil_has_radius_two():
    """"the memory needed ... is one line outward less in each direction" than the public
    goods game's three: flipping any site farther than Manhattan distance 2 from x changes nothing."""
    L = 12
    tab = orc.pd_accept_table(*GEN, 0.5)
    lat = wl.random_lattice(L, 0.5, seed=77)
    i, j = 6, 5
    base = [orc.pd_flip_threshold(lat, tab, i, j, d) for d in range(4)]
    touched = set()
    for a in range(L):
        for b in range(L):
            dist = min(abs(a - i), L - abs(a - i)) + min(abs(b - j), L - abs(b - j))
            lat2 = lat.copy(); lat2[a, b] ^= 1
            now = [orc.pd_flip_threshold(lat2, tab, i, j, d) for d in range(4)]
            if now != base:
                touched.add(dist)
                assert dist <= 2, (a, b)
    assert touched == {0, 1, 2}


def test_step_is_strict_and_directions_match_numpy_indexing():
    tab = orc.pd_accept_table(*GEN, 0.7)
    rng = np.random.default_rng(3)
    n = 0
    for L in (4, 8, 12):
        lat = wl.random_lattice(L, 0.5, seed=L + 40)
        for _ in range(60):
            i, j = (int(v) for v in rng.integers(0, L, size=2))
            for d in range(4):
                sx, sy = int(lat[i, j]), int(lat[(i + DI[d]) % L, (j + DJ[d]) % L])
                thr = orc.pd_flip_threshold(lat, tab, i, j, d)
                if sx == sy:
                    assert thr == 0 and orc.pd_step_given_draw(lat, tab, i, j, d, 0) == sx
                    continue
                if thr > 0:
                    assert orc.pd_step_given_draw(lat, tab, i, j, d, thr - 1) == sy
                assert orc.pd_step_given_draw(lat, tab, i, j, d, thr) == sx
                n += 1
    assert n > 200


def test_schedule_invariants():
    """Absorbing states, changes only at sites of the phase's class, visiting-order independence,
    composition (a,b)+(a+b,c) == (a,b+c), counts are recounts."""
    L = 16
    for v in (0, 1):
        lat = np.full((L, L), v, dtype=np.uint8)
        c = orc.pd_sweep(lat, R, S, T, P, 0.1, 3, n_mcs=5)
        assert (lat == v).all() and (c == v * L * L).all()
    tab = orc.pd_accept_table(R, S, T, P, 0.3)
    lat0 = wl.random_lattice(L, 0.5, seed=9)
    for c in (0, 5, 15):
        a, b = lat0.copy(), lat0.copy()
        da = orc.pd_phase(a, tab, 11, 2, 7, c, visit=0)
        db = orc.pd_phase(b, tab, 11, 2, 7, c, visit=1)
        assert np.array_equal(a, b) and da == db == int(a.sum()) - int(lat0.sum())
        changed = np.argwhere(a != lat0)
        assert all(i % 4 == c >> 2 and j % 4 == c & 3 for i, j in changed)
    one = lat0.copy()
    c_one = orc.pd_sweep(one, R, S, T, P, 0.3, 21, orc.ORDER_IID, 5, 9)
    two = lat0.copy()
    c1 = orc.pd_sweep(two, R, S, T, P, 0.3, 21, orc.ORDER_IID, 5, 4)
    c2 = orc.pd_sweep(two, R, S, T, P, 0.3, 21, orc.ORDER_IID, 9, 5)
    assert np.array_equal(one, two) and np.array_equal(np.concatenate([c1, c2]), c_one)
    assert int(c_one[-1]) == int(one.sum())


def test_dilemma_strength_decides_the_outcome():
    """No dilemma (T < R: cooperation pays at equal neighbourhoods) -> cooperators take over; a strong
    temptation (T = 2 R) -> they die out.  Statistics only (the paper prints no number for this game)."""
    L = 48
    lat = orc.init(L, 0.5, 4)
    c = orc.pd_sweep(lat, 1.0, 0.0, 0.7, 0.0, 0.1, 4, n_mcs=400)
    assert int(c[-1]) > 0.98 * L * L
    lat = orc.init(L, 0.5, 4)
    c = orc.pd_sweep(lat, 1.0, 0.0, 2.0, 0.0, 0.1, 4, n_mcs=400)
    assert int(c[-1]) == 0
