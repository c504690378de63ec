"""Pins for the static parts of the oracle: Philox, payoffs, Fermi table.

Each test checks oracle/ against something other than itself: published
known-answer vectors, closed forms derived by hand from Eqs. (1)-(3) of the
paper, or a 60-digit evaluation of Eq. (3).
"""
from decimal import Decimal, getcontext
from pathlib import Path

import numpy as np
import pytest

import oracle as orc
import workloads as wl

GOLDEN = Path(__file__).parent / "golden"


# ------------------------------------------------------------------ Philox (D1)
def test_philox_known_answers():
    rows = [l.split() for l in (GOLDEN / "philox4x32_10_kat.txt").read_text().splitlines()
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for row in rows:
        v = [int(x, 16) for x in row]
        out = orc.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_philox_counter_and_key_sensitivity():
    """A dropped counter word or key word would make some of these collide."""
    base = orc.philox4x32_10([1, 2, 3, 4], [5, 6]).tolist()
    seen = {tuple(base)}
    for pos in range(4):
        c = [1, 2, 3, 4]
        c[pos] ^= 1
        seen.add(tuple(orc.philox4x32_10(c, [5, 6]).tolist()))
    for pos in range(2):
        k = [5, 6]
        k[pos] ^= 1
        seen.add(tuple(orc.philox4x32_10([1, 2, 3, 4], k).tolist()))
    assert len(seen) == 7


# ------------------------------------------------------------------ payoffs (D2)
R = 4.0


def _lat(L, fill):
    return np.full((L, L), fill, dtype=np.uint8)


def _check(lat, i, j, A, r=R):
    assert orc.A(lat, i, j) == A
    s = int(lat[i % lat.shape[0], j % lat.shape[0]])
    # Pi = (r/5) A - 5 s  follows from Eqs. (1)-(2) with c=1, G=5
    assert orc.payoff_literal(lat, i, j, r) == pytest.approx(r * A / 5.0 - 5.0 * s, abs=1e-12)


def test_payoff_all_C_and_all_D():
    """All-C: every group has N_C=5: Pi = 5 (r*5/5 - 1) = 5(r-1); all-D: 0 (north_star)."""
    for r in (3.5, 4.0, 5.5):
        assert orc.payoff_literal(_lat(8, 1), 3, 3, r) == pytest.approx(5 * (r - 1), abs=1e-12)
        assert orc.payoff_literal(_lat(8, 0), 3, 3, r) == 0.0
    _check(_lat(8, 1), 0, 0, 25)
    _check(_lat(8, 0), 7, 7, 0)


def test_payoff_lone_cooperator():
    """Lone C in a D sea.  Each of C's 5 groups holds exactly one cooperator: A=5, Pi=r-5.
    A nearest D neighbour y shares 2 groups with C (centred on y and on C): A=2, Pi=2r/5.
    A diagonal D shares 2 groups (centred on the two common neighbours): A=2.
    An axial distance-2 D shares 1 group (centred on the site between): A=1, Pi=r/5."""
    lat = _lat(12, 0)
    lat[5, 5] = 1
    _check(lat, 5, 5, 5)
    assert orc.payoff_literal(lat, 5, 5, R) == pytest.approx(-1.0)
    for di, dj in ((1, 0), (-1, 0), (0, 1), (0, -1), (1, 1), (1, -1), (-1, 1), (-1, -1)):
        _check(lat, 5 + di, 5 + dj, 2)
    assert orc.payoff_literal(lat, 5, 6, R) == pytest.approx(1.6)
    for di, dj in ((2, 0), (-2, 0), (0, 2), (0, -2)):
        _check(lat, 5 + di, 5 + dj, 1)
    assert orc.payoff_literal(lat, 7, 5, R) == pytest.approx(0.8)
    for di, dj in ((3, 0), (2, 1), (1, 2), (0, 3), (2, 2)):
        _check(lat, 5 + di, 5 + dj, 0)  # beyond the radius-2 reach of a payoff


def test_payoff_lone_defector():
    """Lone D in a C sea: complement of the above: D A=25-5=20 Pi=4r; nearest C A=23;
    axial distance-2 C A=24."""
    lat = _lat(12, 1)
    lat[5, 5] = 0
    _check(lat, 5, 5, 20)
    assert orc.payoff_literal(lat, 5, 5, R) == pytest.approx(16.0)
    _check(lat, 4, 5, 23)
    assert orc.payoff_literal(lat, 4, 5, R) == pytest.approx(13.4)
    _check(lat, 5, 7, 24)
    assert orc.payoff_literal(lat, 5, 7, R) == pytest.approx(14.2)


def test_payoff_straight_interface():
    """Columns j<6 C, 6<=j<12 D (L=24 so the second interface is far).
    Boundary C (j=5): own 5 + nearest {up,down,left}=3 x2 + diagonals {left-up,left-down}=2 x2
    + distance-2 {up2,down2,left2}=3 x1 = 18, Pi = 18r/5-5 = 9.4.
    Boundary D (j=6): nearest {left}=1 x2 + diagonals {left-up,left-down}=2 x2 + distance-2
    {left2}=1 = 7, Pi=5.6.  Next D column (j=7): only left2 is C: A=1."""
    lat = _lat(24, 0)
    lat[:, :6] = 1
    _check(lat, 10, 5, 18)
    assert orc.payoff_literal(lat, 10, 5, R) == pytest.approx(9.4)
    _check(lat, 10, 6, 7)
    assert orc.payoff_literal(lat, 10, 6, R) == pytest.approx(5.6)
    _check(lat, 10, 7, 1)
    # transposed operand check: a horizontal interface gives the same numbers along i
    _check(np.ascontiguousarray(lat.T), 5, 10, 18)
    _check(np.ascontiguousarray(lat.T), 6, 10, 7)


def test_payoff_checkerboard_and_block():
    """Checkerboard: C site: own 5 + diagonals 4x2 + distance-2 4x1 = 17 (Pi=8.6); D site:
    nearest 4x2 = 8 (Pi=6.4).  2x2 C block: each C: 5 + 2 nearest x2 + 1 diagonal x2 = 11
    (Pi=3.8); D right of the top-right C: nearest 1 x2 + diagonal 1 x2 + distance-2 1 = 5 (Pi=4)."""
    cb = wl.checkerboard_lattice(8)
    ci, cj = (0, 1) if cb[0, 1] == 1 else (0, 0)
    _check(cb, ci, cj, 17)
    assert orc.payoff_literal(cb, ci, cj, R) == pytest.approx(8.6)
    _check(cb, ci, cj + 1, 8)
    assert orc.payoff_literal(cb, ci, cj + 1, R) == pytest.approx(6.4)
    lat = _lat(12, 0)
    lat[4:6, 4:6] = 1
    for i in (4, 5):
        for j in (4, 5):
            _check(lat, i, j, 11)
    assert orc.payoff_literal(lat, 4, 4, R) == pytest.approx(3.8)
    _check(lat, 4, 6, 5)
    assert orc.payoff_literal(lat, 4, 6, R) == pytest.approx(4.0)


def _A_weight_form(lat):
    """A_x = 5 s_x + 2*(4 nearest) + 2*(4 diagonal) + 1*(4 axial distance-2): counts, for each
    site w, the pairs (group centre z in cross(x), member w in cross(z)); derived by hand in
    DESIGN.md.  Weights sum to 25."""
    s = lat.astype(np.int64)
    sh = lambda a, b: np.roll(np.roll(s, a, axis=0), b, axis=1)
    near = sh(1, 0) + sh(-1, 0) + sh(0, 1) + sh(0, -1)
    diag = sh(1, 1) + sh(1, -1) + sh(-1, 1) + sh(-1, -1)
    ax2 = sh(2, 0) + sh(-2, 0) + sh(0, 2) + sh(0, -2)
    return 5 * s + 2 * near + 2 * diag + ax2


@pytest.mark.parametrize("L", [4, 8, 12, 20])
def test_A_matches_weight_form_on_random_lattices(L):
    """Includes L=4, where x+2e and x-2e coincide under the periodic wrap."""
    for seed in range(4):
        lat = wl.random_lattice(L, 0.5, 100 * L + seed)
        Aw = _A_weight_form(lat)
        for i in range(L):
            for j in range(L):
                assert orc.A(lat, i, j) == Aw[i, j]


def test_payoff_group_centric_accumulation():
    """Brute force, written the other way round: loop over GROUPS, hand every
    member its Eq. (1)/(2) share, and accumulate per player.  A transposed operand or a dropped
    group in the oracle's player-centric gather would break this."""
    L, r = 10, 3.8
    lat = wl.random_lattice(L, 0.4, 7)
    total = np.zeros((L, L))
    off = [(0, 0), (-1, 0), (1, 0), (0, -1), (0, 1)]
    for zi in range(L):
        for zj in range(L):
            members = [((zi + a) % L, (zj + b) % L) for a, b in off]
            NC = sum(int(lat[m]) for m in members)
            for m in members:
                total[m] += r * 1.0 * NC / 5.0 - (1.0 if lat[m] else 0.0)
    for i in range(L):
        for j in range(L):
            assert orc.payoff_literal(lat, i, j, r) == pytest.approx(total[i, j], abs=1e-12)


def test_defection_gain_is_G_minus_r():
    """with the others fixed, switching x from C to D changes its own payoff by
    5c - r c (it saves 5 contributions and loses r/5 from each of its 5 groups), positive iff
    r < G = 5 -- the social dilemma and the well-mixed threshold r = G."""
    for r in (3.0, 4.9, 5.0, 6.0):
        lat = wl.random_lattice(9, 0.5, 3)
        lat[4, 4] = 1
        pc = orc.payoff_literal(lat, 4, 4, r)
        lat[4, 4] = 0
        pd = orc.payoff_literal(lat, 4, 4, r)
        assert pd - pc == pytest.approx(5.0 - r, abs=1e-12)


def test_group_count_includes_centre_and_four_neighbours():
    lat = _lat(8, 0)
    lat[3, 3] = 1
    assert orc.group_count(lat, 3, 3) == 1
    for di, dj in ((1, 0), (-1, 0), (0, 1), (0, -1)):
        assert orc.group_count(lat, 3 + di, 3 + dj) == 1
    assert orc.group_count(lat, 4, 4) == 0
    lat[0, 0] = 1  # periodic wrap
    assert orc.group_count(lat, 7, 0) == 1 and orc.group_count(lat, 0, 7) == 1


# ------------------------------------------------------------------ Fermi table (D3)
def _exact_T(r, K, dA, ds):
    getcontext().prec = 60
    z = (Decimal(r) * dA / 5 - 5 * ds) / Decimal(K)
    if z > 200:
        W = Decimal(0)
    else:
        W = 1 / (1 + z.exp())
    v = W * (1 << 32)
    fl = int(v)  # v >= 0
    frac = float(v - fl)
    return min(fl, 0xFFFFFFFF), frac


@pytest.mark.parametrize("r,K", [(4.0, 0.5), (3.8, 0.5), (3.7443, 0.5), (3.98, 0.5), (5.5, 0.5),
                                 (3.70 + (0.1 * 17) / 63.0, 0.5), (4.0, 0.1), (4.0, 2.0)])
def test_table_matches_fermi_formula_at_60_digits(r, K):
    """Eq. (3) PAPER.md:60 evaluated exactly (r, K taken as the doubles they are)."""
    T = orc.accept_table(r, K)
    for ds in (-1, 0, 1):
        for dA in range(-25, 26):
            exact, frac = _exact_T(r, K, dA, ds)
            got = int(T[orc.table_index(dA, ds)])
            if got != exact:
                # double rounding can only matter within ~1e-5 of an integer boundary
                assert abs(got - exact) == 1 and min(frac, 1 - frac) < 1e-4, (dA, ds, got, exact)


def test_table_index_layout():
    assert orc.table_index(-25, -1) == 0
    assert orc.table_index(25, -1) == 50
    assert orc.table_index(0, 0) == 76
    assert orc.table_index(25, 1) == 152


def test_table_facts():
    """S7/S8 and monotonicity: W decreases with Pi_x - Pi_y."""
    r, K = 4.0, 0.5
    T = orc.accept_table(r, K)
    assert T[orc.table_index(0, 0)] == 0x80000000  # tie: W = 1/2
    assert T[orc.table_index(-25, -1)] == 0xFFFFFFFF  # W rounds to 1: clamp (S7)
    assert T[orc.table_index(25, 1)] == 0
    pairs = sorted(((r * dA) / 5.0 - 5.0 * ds, int(T[orc.table_index(dA, ds)]))
                   for ds in (-1, 0, 1) for dA in range(-25, 26))
    for (d0, t0), (d1, t1) in zip(pairs, pairs[1:]):
        assert t1 <= t0 or d1 == d0
    # W(d) + W(-d) = 1
    for ds in (-1, 0, 1):
        for dA in range(-25, 26):
            a = int(T[orc.table_index(dA, ds)])
            b = int(T[orc.table_index(-dA, -ds)])
            if 0 < a < 0xFFFFFFFF and 0 < b < 0xFFFFFFFF:
                assert a + b in (2**32 - 1, 2**32)


def test_table_limits_of_K():
    """K->0: x copies y iff Pi_y > Pi_x; K->infinity: coin flip."""
    r = 4.0
    T = orc.accept_table(r, 1e-3)
    for ds in (-1, 0, 1):
        for dA in range(-25, 26):
            d = (r * dA) / 5.0 - 5.0 * ds
            t = int(T[orc.table_index(dA, ds)])
            if d > 0:
                assert t == 0
            elif d < 0:
                assert t == 0xFFFFFFFF
            else:
                assert t == 0x80000000
    T = orc.accept_table(r, 1e9)
    assert np.all(np.abs(T.astype(np.int64) - 2**31) < 2**31 * 1e-6)


def test_fermi_function_direct():
    """Eq. (3): W = 1/(1+exp((Pi_x-Pi_y)/K)); large Pi_y => W -> 1 (S12)."""
    assert orc.fermi(1.0, 1.0, 0.5) == 0.5
    assert orc.fermi(0.0, 10.0, 0.5) > 0.999999
    assert orc.fermi(10.0, 0.0, 0.5) < 1e-6
    import math
    assert orc.fermi(2.6, 0.0, 0.5) == pytest.approx(1 / (1 + math.exp(5.2)), rel=1e-15)
    # printed-digit check of the lone-D example in SURVEY P3: Delta=2.6, K=.5 -> W=0.00548629889945
    assert orc.fermi(2.6, 0.0, 0.5) == pytest.approx(0.00548629889945, abs=1e-13)


def test_table_consistent_with_literal_payoffs():
    """T/2^32 equals W computed from the two literal 5-group payoffs (not from dA)."""
    r, K = 3.8, 0.5
    T = orc.accept_table(r, K)
    di = [-1, 1, 0, 0]
    dj = [0, 0, -1, 1]
    n = 0
    for seed in range(6):
        L = 12
        lat = wl.random_lattice(L, 0.5, 50 + seed)
        for i in range(L):
            for j in range(L):
                for d in range(4):
                    yi, yj = (i + di[d]) % L, (j + dj[d]) % L
                    if lat[i, j] == lat[yi, yj]:
                        assert orc.flip_threshold(lat, T, i, j, d) == 0
                        continue
                    W = orc.fermi(orc.payoff_literal(lat, i, j, r),
                                  orc.payoff_literal(lat, yi, yj, r), K)
                    assert orc.flip_threshold(lat, T, i, j, d) / 2**32 == pytest.approx(W, abs=1e-9)
                    n += 1
    assert n > 500
