"""Pins for the dynamic parts of the oracle: init, schedule, phases, sweeps.

Independent anchors: exact one-step law on all 2^16 states of the 4x4 torus
(brute force, payoffs accumulated group by group in numpy), invariants the
method guarantees (absorbing states, order independence, composition), binomial
statistics of the draws, and SURVEY.md's advisory third-opinion trajectory.
"""
from pathlib import Path

import numpy as np
import pytest

import oracle as orc
import workloads as wl

GOLDEN = Path(__file__).parent / "golden"


def _golden_p9():
    out = {}
    for line in (GOLDEN / "survey_p9_advisory.txt").read_text().splitlines():
        if not line.strip() or line.startswith("#"):
            continue
        key, *vals = line.split()
        out[key] = vals
    return out


# ------------------------------------------------------------------ init (D4)
def test_init_extremes_are_exact():
    assert orc.count(orc.init(16, 0.0, 5)) == 0
    assert orc.count(orc.init(16, 1.0, 5)) == 256


def test_init_is_bernoulli():
    """PAPER.md:58 'with equal probability': fraction within 5 sigma of rho0; adjacent sites
    uncorrelated; different seeds differ."""
    L = 256
    for rho0 in (0.5, 0.2):
        lat = orc.init(L, rho0, 11)
        n = L * L
        assert abs(orc.count(lat) - rho0 * n) < 5 * np.sqrt(n * rho0 * (1 - rho0))
        a = lat.astype(np.float64) - rho0
        corr = (a * np.roll(a, 1, axis=1)).mean() / (rho0 * (1 - rho0))
        assert abs(corr) < 5 / np.sqrt(n)
    assert np.any(orc.init(32, 0.5, 1) != orc.init(32, 0.5, 2))


def test_init_matches_advisory_first_sites():
    g = _golden_p9()
    lat = orc.init(64, 0.5, 1)
    assert orc.count(lat) == int(g["count0"][0])
    assert "".join(map(str, lat.ravel()[:32])) == g["init_first32"][0]


# ------------------------------------------------------------------ schedule (D5)
def test_phase_classes_iid_and_perm():
    for t in range(50):
        iid = orc.phase_classes(9, t, orc.ORDER_IID)
        assert iid.min() >= 0 and iid.max() < 16
        perm = orc.phase_classes(9, t, orc.ORDER_PERM)
        assert sorted(perm.tolist()) == list(range(16))


def test_phase_classes_iid_uniform():
    """S2: per-site update counts are Binomial(16, 1/16) -- classes uniform over many MCS."""
    counts = np.zeros(16)
    T = 4000
    for t in range(T):
        for c in orc.phase_classes(3, t, orc.ORDER_IID):
            counts[c] += 1
    exp = 16 * T / 16
    chi2 = ((counts - exp) ** 2 / exp).sum()
    assert chi2 < 45  # 15 dof, p ~ 1e-4


def test_phase_classes_perm_uniform_first_position():
    first = np.zeros(16)
    for t in range(3200):
        first[orc.phase_classes(4, t, orc.ORDER_PERM)[0]] += 1
    chi2 = ((first - 200) ** 2 / 200).sum()
    assert chi2 < 45


def test_phase_classes_match_advisory():
    g = _golden_p9()
    assert orc.phase_classes(1, 0, orc.ORDER_IID).tolist() == [int(x) for x in g["iid_classes_t0"]]
    assert orc.phase_classes(1, 0, orc.ORDER_PERM).tolist() == [int(x) for x in g["perm_classes_t0"]]


def test_step_draw_statistics_and_advisory():
    g = _golden_p9()
    d, u = orc.step_draw(1, 0, 0, 0, 0)
    x0, x1 = (int(v, 16) for v in g["step_draw_site0_t0_k0_c0"])
    assert d == x0 >> 30 and u == x1
    dirs = np.zeros(4)
    us = []
    for site in range(4000):
        d, u = orc.step_draw(77, site, 3, 5, 9)
        dirs[d] += 1
        us.append(u / 2**32)
    assert ((dirs - 1000) ** 2 / 1000).sum() < 25  # 3 dof
    assert abs(np.mean(us) - 0.5) < 5 / np.sqrt(12 * 4000)
    # k, c, t and site all enter the counter (S3)
    base = orc.step_draw(77, 10, 3, 5, 9)
    assert len({base, orc.step_draw(77, 11, 3, 5, 9), orc.step_draw(77, 10, 4, 5, 9),
                orc.step_draw(77, 10, 3, 6, 9), orc.step_draw(77, 10, 3, 5, 10),
                orc.step_draw(78, 10, 3, 5, 9)}) == 6


# ------------------------------------------------------------------ 4x4 brute force (P5)
def _all_4x4_states():
    idx = np.arange(1 << 16, dtype=np.uint32)
    bits = ((idx[:, None] >> np.arange(16)[None, :]) & 1).astype(np.uint8)
    return bits.reshape(-1, 4, 4)


def _payoffs_group_centric(S, r):
    """S: [n,4,4].  For every group (centre z) compute N_C and add each member's Eq. (1)/(2)
    share to that member's total."""
    s = S.astype(np.float64)
    N = s.copy()
    for ax, sh in ((1, 1), (1, -1), (2, 1), (2, -1)):
        N += np.roll(s, sh, axis=ax)
    total = np.zeros_like(s)
    share = r * N / 5.0  # what the group centred on z pays each member, before costs
    # member = centre + offset  <=>  total[m] += share[m - offset]
    for ax, sh in ((None, 0), (1, 1), (1, -1), (2, 1), (2, -1)):
        total += share if ax is None else np.roll(share, sh, axis=ax)
    total -= 5.0 * s  # a cooperator pays c = 1 in each of its 5 groups
    return total


@pytest.mark.parametrize("r,K", [(4.0, 0.5), (3.8, 0.5)])
def test_exact_one_step_law_on_4x4_torus(r, K):
    """For all 2^16 states, all 16 focal sites and all 4 directions the oracle's acceptance
    threshold equals Eq. (3) with brute-force payoffs, within 2^-32 (plus double rounding).
    L=4 also exercises the wrap where x+2e == x-2e."""
    S = _all_4x4_states()
    T = orc.accept_table(r, K)
    thr = orc.flip_thresholds_batch(S, T).astype(np.float64) / 2**32  # [n,4,4,4]
    P = _payoffs_group_centric(S, r)
    s = S.astype(np.int64)
    shifts = [(1, 1), (1, -1), (2, 1), (2, -1)]  # dir 0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1)
    for d, (ax, sh) in enumerate(shifts):
        Py = np.roll(P, sh, axis=ax)
        sy = np.roll(s, sh, axis=ax)
        W = 1.0 / (1.0 + np.exp((P - Py) / K))
        want = np.where(sy != s, W, 0.0)
        err = np.abs(thr[..., d] - want)
        assert err.max() < 2.0**-32 + 1e-12, (d, err.max())
        assert np.all(thr[..., d][sy == s] == 0)


def test_empirical_flip_frequency_matches_law():
    """Run the real phase stepping (Philox draws) on L=4 many times from the same state and
    compare the flip frequency of each site with 1/4 sum_dir T/2^32 within binomial error."""
    r, K = 4.0, 0.5
    T = orc.accept_table(r, K)
    lat0 = np.array([[1, 1, 0, 0], [1, 0, 0, 1], [0, 0, 1, 1], [0, 1, 1, 0]], dtype=np.uint8)
    thr = orc.flip_thresholds_batch(lat0[None], T)[0].astype(np.float64) / 2**32
    p = thr.mean(axis=-1)  # [4,4]
    n = 6000
    flips = np.zeros((4, 4))
    for t in range(n):
        for c in range(16):
            lat = lat0.copy()
            orc.phase(lat, T, 12345, t, 0, c)
            i, j = c >> 2, c & 3
            changed = lat != lat0
            assert changed.sum() <= 1 and (changed.sum() == 0 or changed[i, j])
            flips[i, j] += changed[i, j]
    sigma = np.sqrt(n * p * (1 - p)) + 1e-9
    assert np.all(np.abs(flips - n * p) < 5 * sigma + 1)
    assert flips.sum() > 100


# ------------------------------------------------------------------ invariants
def test_absorbing_states_stay_absorbing():
    """PAPER.md:111 (absorbing phase): all-D and all-C never change under any schedule."""
    for fill in (0, 1):
        for mode in (orc.ORDER_IID, orc.ORDER_PERM):
            lat = np.full((16, 16), fill, dtype=np.uint8)
            counts, _ = orc.sweep(lat, 3.9, 0.5, 4, mode, 0, 20)
            assert np.all(lat == fill) and np.all(counts == fill * 256)
        lat = np.full((16, 16), fill, dtype=np.uint8)
        counts = orc.rs_sweep(lat, 3.9, 0.5, 4, 0, 5)
        assert np.all(lat == fill) and np.all(counts == fill * 256)


def test_order_independence_within_a_phase():
    """S1/P6: raster, reverse and shuffled visiting orders give identical lattices, and only
    sites of the active class can change."""
    L = 24
    T = orc.accept_table(4.0, 0.5)
    rng = np.random.default_rng(0)
    for trial in range(12):
        lat0 = wl.random_lattice(L, 0.5, trial)
        c = int(rng.integers(16))
        k = int(rng.integers(16))
        a, b, d = lat0.copy(), lat0.copy(), lat0.copy()
        da = orc.phase(a, T, 5, trial, k, c, visit=0)
        db = orc.phase(b, T, 5, trial, k, c, visit=1)
        perm = rng.permutation((L // 4) ** 2).astype(np.uint32)
        dd = orc.phase(d, T, 5, trial, k, c, visit=2, perm=perm)
        e = lat0.copy()
        de = orc.phase(e, T, 5, trial, k, c, visit=0, n_threads=3)
        assert np.array_equal(a, b) and np.array_equal(a, d) and np.array_equal(a, e)
        assert da == db == dd == de == int(a.sum()) - int(lat0.sum())
        changed = np.argwhere(a != lat0)
        assert all(4 * (i % 4) + (j % 4) == c for i, j in changed)


def test_read_stencil_radius_is_three():
    """a step at x needs strategies at most three lines outward.  Flipping any
    site farther than Manhattan distance 3 from x must never change the outcome at x, and some
    site at distance exactly 3 must matter."""
    L = 16
    T = orc.accept_table(4.0, 0.5)
    lat = wl.random_lattice(L, 0.5, 21)
    x = (8, 8)
    matters = set()
    for seed in range(40):
        lat = wl.random_lattice(L, 0.5, seed)
        for d in range(4):
            base = orc.flip_threshold(lat, T, x[0], x[1], d)
            for i in range(L):
                for j in range(L):
                    dist = min(abs(i - 8), L - abs(i - 8)) + min(abs(j - 8), L - abs(j - 8))
                    if dist == 0:
                        continue
                    lat[i, j] ^= 1
                    if orc.flip_threshold(lat, T, x[0], x[1], d) != base:
                        matters.add(dist)
                        assert dist <= 3
                    lat[i, j] ^= 1
    assert 3 in matters


def test_composition_and_trace_convention():
    """P7/D7: (a,b) then (a+b,c) == (a,b+c); counts[m] is the recount after MCS t_begin+m."""
    L = 32
    for mode in (orc.ORDER_IID, orc.ORDER_PERM):
        one = orc.init(L, 0.5, 3)
        two = one.copy()
        c_all, snaps = orc.sweep(one, 3.9, 0.5, 3, mode, 0, 12, snap_every=1)
        c_a, _ = orc.sweep(two, 3.9, 0.5, 3, mode, 0, 5)
        c_b, _ = orc.sweep(two, 3.9, 0.5, 3, mode, 5, 7)
        assert np.array_equal(one, two)
        assert np.array_equal(c_all, np.concatenate([c_a, c_b]))
        assert [int(s.sum()) for s in snaps] == [int(c) for c in c_all]


def test_mcs_is_L2_elementary_steps():
    """one MCS = L^2 elementary steps = 16 phases x L^2/16 sites."""
    L = 12
    T = orc.accept_table(4.0, 0.5)
    lat = wl.random_lattice(L, 0.5, 1)
    sites = 0
    for k in range(16):
        sites += (L // 4) ** 2
        orc.phase(lat, T, 1, 0, k, k)
    assert sites == L * L


def test_config1_advisory_trajectory():
    """SURVEY.md P9 advisory values (independent restatements at survey time)."""
    g = _golden_p9()
    for mode, key in ((orc.ORDER_IID, "iid_counts_after_mcs"), (orc.ORDER_PERM, "perm_counts_after_mcs")):
        lat = orc.init(64, 0.5, 1)
        counts, _ = orc.sweep(lat, 4.0, 0.5, 1, mode, 0, 1000)
        for item in g[key]:
            m, v = item.split(":")
            assert int(counts[int(m) - 1]) == int(v)


def test_pack_unpack_bits_layout():
    """site (i,j) is bit (j&31) of little-endian word i*(L/32) + (j>>5)."""
    L = 64
    lat = np.zeros((L, L), dtype=np.uint8)
    lat[3, 37] = 1
    w = orc.pack_bits(lat)
    assert w[3, 1] == 1 << 5 and w.sum() == 1 << 5
    lat = wl.random_lattice(L, 0.5, 8)
    assert np.array_equal(orc.unpack_bits(orc.pack_bits(lat), L), lat)
    # same bytes as numpy's little-endian bit packing
    assert np.array_equal(orc.pack_bits(lat).view(np.uint8).reshape(L, L // 8),
                          np.packbits(lat, axis=1, bitorder="little"))


def test_rs_sweep_counts_and_site_coverage():
    """D8: random sequential: counts are recounts; one MCS is L^2 picks of a uniformly drawn focal
    site, so a given site is never picked with probability (1 - 1/N)^N ~ 1/e.
    Observable through the dynamics: at r = 4, K = 1e-3 a lone cooperator in a defector sea
    (payoff r - 5 = -1 against its neighbours' 2r/5 = 1.6) turns defector the first
    time it is the focal site, whatever direction it draws, and no defector ever adopts from it.
    So the lone cooperators that survive one MCS are exactly the never-picked ones."""
    L = 32
    lat = orc.init(L, 0.5, 2)
    before = lat.copy()
    counts = orc.rs_sweep(lat, 4.0, 0.5, 2, 0, 3)
    assert int(counts[-1]) == int(lat.sum())
    assert np.any(lat != before)
    L, spacing = 200, 5
    survivors, n_lone = 0, 0
    for seed in (3, 4, 5):
        lat = np.zeros((L, L), dtype=np.uint8)
        lat[2::spacing, 2::spacing] = 1          # isolated: 5 apart, neighbourhoods do not touch
        lone = lat.copy()
        n_lone += int(lone.sum())
        c = orc.rs_sweep(lat, 4.0, 1e-3, seed, 0, 1)
        assert not np.any(lat & (1 - lone)), "a defector adopted cooperation from a poorer neighbour"
        assert int(c[0]) == int(lat.sum())
        survivors += int(lat.sum())
    p = (1.0 - 1.0 / (L * L)) ** (L * L)         # = 0.36787..., 1/e to four digits
    sigma = (n_lone * p * (1 - p)) ** 0.5
    assert abs(survivors - n_lone * p) < 4 * sigma, (survivors, n_lone * p, sigma)
    assert abs(1 - survivors / n_lone - (1 - np.exp(-1))) < 0.03   # visited fraction ~ 1 - 1/e


def test_step_accepts_strictly_below_the_threshold_in_every_direction():
    """D3 / D6: x adopts s_y iff u < T (strict), with y the neighbour in direction
    0:(i-1,j) 1:(i+1,j) 2:(i,j-1) 3:(i,j+1).  T comes from orc_flip_threshold, whose direction
    table the 4x4 brute force pins; s_y is read here by numpy indexing, so the separate
    direction table inside orc_step_given_draw is checked against both.  P(u < T) = T / 2^32
    is Eq. (3) only with the strict compare: `<=` would pass every other pin."""
    di, dj = (-1, 1, 0, 0), (0, 0, -1, 1)
    table = orc.accept_table(3.9, 0.5)
    rng = np.random.default_rng(12)
    n_checked = 0
    for L, p in ((8, 0.5), (12, 0.3), (4, 0.5)):
        for rep in range(6):
            lat = wl.random_lattice(L, p, seed=100 * L + rep)
            for _ in range(40):
                i, j = (int(v) for v in rng.integers(0, L, size=2))
                for d in range(4):
                    sx = int(lat[i, j])
                    sy = int(lat[(i + di[d]) % L, (j + dj[d]) % L])
                    T = orc.flip_threshold(lat, table, i, j, d)
                    if sx == sy:
                        assert T == 0
                        for u in (0, 1, 0x7FFFFFFF, 0xFFFFFFFF):
                            assert orc.step_given_draw(lat, table, i, j, d, u) == sx
                        continue
                    assert T == int(table[orc.table_index(orc.A(lat, i, j) - orc.A(lat, (i + di[d]) % L, (j + dj[d]) % L),
                                                          sx - sy)])
                    if T > 0:
                        assert orc.step_given_draw(lat, table, i, j, d, T - 1) == sy, "u = T - 1 must be accepted"
                        assert orc.step_given_draw(lat, table, i, j, d, 0) == sy
                    assert orc.step_given_draw(lat, table, i, j, d, T) == sx, "u = T must be rejected (strict <)"
                    assert orc.step_given_draw(lat, table, i, j, d, 0xFFFFFFFF) == sx
                    n_checked += 1
    assert n_checked > 500
