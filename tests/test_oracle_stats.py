"""Statistical pins of the oracle against values the paper prints.

These are physics checks: a dropped payoff term, a wrong sign in the Fermi
exponent or a biased schedule moves the stationary cooperator density far
outside the tolerances below (e.g. the PERM schedule alone shifts rho_C(3.98)
by +0.01, a sign error drives the lattice to an absorbing state).
"""
import numpy as np

import oracle as orc

K = 0.5


def _stationary(L, r, mode, n_mcs, discard, seed, n_threads=4):
    lat = orc.init(L, 0.5, seed)
    if mode == "rs":
        c = orc.rs_sweep(lat, r, K, seed, 0, n_mcs)
    else:
        c, _ = orc.sweep(lat, r, K, seed, mode, 0, n_mcs, n_threads=n_threads)
    return c[discard:].mean() / (L * L)


def test_rho_half_at_r_3_98_sublattice_iid():
    """'K = 0.5 and r = 3.98 at which the fraction of cooperators in the
    stationary state is rho_C = 0.5'.  L=128, 3000 MCS, first 1500 discarded; the run-to-run
    scatter at this size is ~0.005."""
    rho = _stationary(128, 3.98, orc.ORDER_IID, 3000, 1500, 7)
    assert abs(rho - 0.5) < 0.015


def test_rho_half_at_r_3_98_random_sequential():
    rho = _stationary(128, 3.98, "rs", 2500, 1200, 7)
    assert abs(rho - 0.5) < 0.015


def test_extinction_below_threshold_and_full_cooperation_above():
    """cooperators survive only for r > 3.74 (r_c = 3.7443)
    inset: at large r the other absorbing phase (all C).  Both schedules."""
    L = 64
    for mode in (orc.ORDER_IID, "rs"):
        lat = orc.init(L, 0.5, 3)
        if mode == "rs":
            c = orc.rs_sweep(lat, 3.5, K, 3, 0, 400)
        else:
            c, _ = orc.sweep(lat, 3.5, K, 3, mode, 0, 400)
        assert c[-1] == 0
    lat = orc.init(L, 0.5, 3)
    c, _ = orc.sweep(lat, 6.0, K, 3, orc.ORDER_IID, 0, 2500)
    assert c[-1] == L * L


def test_cooperators_survive_above_threshold():
    """r = 3.9 > r_c: the mixed C+D phase."""
    rho = _stationary(96, 3.9, orc.ORDER_IID, 2000, 1000, 5)
    assert 0.3 < rho < 0.55
