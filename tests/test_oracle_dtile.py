"""Pins for the oracle's double-tiling schedule (the paper's own parallel scheme).

The elementary step it performs (``step_given_draw``) and Philox are pinned elsewhere (4x4 brute
force, known answers).  What is pinned here is the schedule around them: the geometry the paper
states (4x4 domains, four types in 2x2 order, same-type domains not sharing "a player or even a
border", L divisible by 8), the readings T1-T4 (16 picks per domain and part = L^2 steps per MCS,
the draw fields, sequential picks), the invariants the scheme guarantees (a part changes only
domains of its type; any visiting order of the domains gives the same lattice; absorbing states),
and the statistics the paper validates it with (rho_C(3.98) = 0.5).
"""
import numpy as np
import pytest

import oracle as orc


def _torus_dist(a, b, L):
    d = abs(a - b)
    return min(d, L - d)


def test_domain_types_follow_fig2():
    """types alternate 1,2,1,2,... along one line of domains and 3,4,3,4,... along the
    next; domains of a type share neither a player nor a border."""
    L = 32
    M = L // 4
    types = np.array([[orc.dtile_type(I, J) for J in range(M)] for I in range(M)])
    assert list(types[0, :4]) == [0, 1, 0, 1] and list(types[1, :4]) == [2, 3, 2, 3]
    for q in range(4):
        assert (types == q).sum() == L * L // 64
    # nearest sites of two different same-type domains are 5 apart in at least one axis: a 4-site gap
    doms = [(I, J) for I in range(M) for J in range(M) if types[I, J] == 0]
    for (I, J) in doms:
        for (I2, J2) in doms:
            if (I, J) == (I2, J2):
                continue
            gi = min(_torus_dist(4 * I + a, 4 * I2 + b, L) for a in range(4) for b in range(4))
            gj = min(_torus_dist(4 * J + a, 4 * J2 + b, L) for a in range(4) for b in range(4))
            assert max(gi, gj) >= 5


def test_L_must_be_divisible_by_8():
    """PAPER.md:83,93."""
    lat = orc.init(12, 0.5, 1)
    with pytest.raises(ValueError):
        orc.sweep(lat, 4.0, 0.5, 1, order_mode=orc.ORDER_DTILE, n_mcs=1)
    orc.sweep(orc.init(8, 0.5, 1), 4.0, 0.5, 1, order_mode=orc.ORDER_DTILE, n_mcs=1)


def test_draw_fields_and_uniformity():
    """T2: the draw of pick p of domain d in MCS t is Philox(ctr=(d,t,p,5)); the focal site is
    uniform over the 16 sites of the domain and the direction over 4."""
    seed = 0x1234567890ABCDEF
    key = [seed & 0xFFFFFFFF, seed >> 32]
    hist = np.zeros((4, 4, 4), dtype=np.int64)
    n = 0
    for d in range(40):
        for t in (0, 7):
            for p in range(16):
                a, b, di, u = orc.dtile_draw(seed, d, t, p)
                x = orc.philox4x32_10([d, t, p, 5], key)
                assert (a, b, di, u) == (int(x[0]) >> 30, (int(x[0]) >> 28) & 3, int(x[2]) >> 30, int(x[1]))
                hist[a, b, di] += 1
                n += 1
    expect = n / 64.0
    chi2 = ((hist - expect) ** 2 / expect).sum()
    assert chi2 < 120.0  # 63 degrees of freedom: mean 63, sigma 11


def _by_hand(lat, table, seed, t, q):
    """Part q replayed pick by pick in Python from the pinned elementary step."""
    L = lat.shape[0]
    M = L // 4
    n_steps = 0
    for I in range(M):
        for J in range(M):
            if 2 * (I & 1) + (J & 1) != q:
                continue
            for p in range(16):
                a, b, di, u = orc.dtile_draw(seed, I * M + J, t, p)
                i, j = 4 * I + a, 4 * J + b
                lat[i, j] = orc.step_given_draw(lat, table, i, j, di, u)
                n_steps += 1
    return n_steps


def test_sweep_is_four_parts_of_sequential_picks_and_L2_steps():
    """T1, T4 and PAPER.md:65,75: one MCS = parts 1,2,3,4 in turn = L^2 elementary steps."""
    L, r, K, seed = 16, 3.9, 0.5, 99
    table = orc.accept_table(r, K)
    lat = orc.init(L, 0.5, seed)
    ref = lat.copy()
    counts, _ = orc.sweep(lat, r, K, seed, order_mode=orc.ORDER_DTILE, t_begin=3, n_mcs=3)
    for m in range(3):
        n = sum(_by_hand(ref, table, seed, 3 + m, q) for q in range(4))
        assert n == L * L
        assert int(counts[m]) == int(ref.sum())
    assert np.array_equal(lat, ref)
    assert not np.array_equal(lat, orc.init(L, 0.5, seed))  # something happened


def test_part_changes_only_its_type_and_any_domain_order_agrees():
    L, r, K, seed = 64, 4.0, 0.5, 5
    table = orc.accept_table(r, K)
    base = orc.init(L, 0.5, seed)
    ii, jj = np.meshgrid(np.arange(L), np.arange(L), indexing="ij")
    dtype = 2 * ((ii >> 2) & 1) + ((jj >> 2) & 1)
    for q in range(4):
        a, b, c = base.copy(), base.copy(), base.copy()
        da = orc.dtile_part(a, table, seed, 1, q, visit=0)
        db = orc.dtile_part(b, table, seed, 1, q, visit=1)
        dc = orc.dtile_part(c, table, seed, 1, q, visit=0, n_threads=3)
        assert np.array_equal(a, b) and np.array_equal(a, c) and da == db == dc
        changed = a != base
        assert changed.any() and np.all(dtype[changed] == q)
        assert da == int(a.sum()) - int(base.sum())


def test_composition_and_absorbing_states():
    L, r, K, seed = 32, 3.8, 0.5, 21
    a = orc.init(L, 0.5, seed)
    b = a.copy()
    ca, _ = orc.sweep(a, r, K, seed, order_mode=orc.ORDER_DTILE, t_begin=0, n_mcs=7)
    c1, _ = orc.sweep(b, r, K, seed, order_mode=orc.ORDER_DTILE, t_begin=0, n_mcs=3)
    c2, _ = orc.sweep(b, r, K, seed, order_mode=orc.ORDER_DTILE, t_begin=3, n_mcs=4)
    assert np.array_equal(a, b) and list(ca) == list(c1) + list(c2)
    for rho0, n in ((0.0, 0), (1.0, L * L)):
        z = orc.init(L, rho0, seed)
        c, _ = orc.sweep(z, r, K, seed, order_mode=orc.ORDER_DTILE, n_mcs=5)
        assert all(int(v) == n for v in c)


def test_stationary_density_at_r398_is_one_half():
    """at K = 0.5 and r = 3.98 'the fraction of cooperators in the stationary state
    is rho_C = 0.5' -- the value the paper's own schedule was benchmarked at."""
    L = 120
    lat = orc.init(L, 0.5, 3)
    c, _ = orc.sweep(lat, 3.98, 0.5, 3, order_mode=orc.ORDER_DTILE, n_mcs=1500)
    rho = c[500:].mean() / (L * L)
    assert abs(rho - 0.5) < 0.02
