"""Seeded, synthetic workload definitions shared by tests/, bench.py and smoke().

This module holds NONE of the method's arithmetic: no Philox, no payoff, no
acceptance table, no schedule.  It only names the five BASELINE.json configs
("each player ... C or D with equal probability", PAPER.md:113,119
for the lattice sizes and K=0.5) and makes arbitrary seeded lattices with
numpy's own generator for tests that start from a given state.  The Philox
Bernoulli initial condition is part of the method
and is implemented independently by oracle/ and by the CUDA library.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Tuple

import numpy as np

K_DEFAULT = 0.5


@dataclass(frozen=True)
class Config:
    name: str
    L: int
    rs: Tuple[float, ...]       # one r per lattice
    seeds: Tuple[int, ...]      # one seed per lattice
    n_mcs: int
    K: float = K_DEFAULT
    rho0: float = 0.5
    snap_every: int = 0
    note: str = ""

    @property
    def batch(self) -> int:
        return len(self.rs)

    @property
    def sites(self) -> int:
        return self.L * self.L


def config1() -> Config:
    """BASELINE.json configs[0]: L=64, r=4.0, seed 1, 1000 MCS, lattice every 100 MCS."""
    return Config("C1_L64", 64, (4.0,), (1,), 1000, snap_every=100)


def config2_rs() -> Tuple[float, ...]:
    lo = tuple(round(3.60 + 0.05 * a, 2) for a in range(9))     # 3.60 .. 4.00
    hi = (5.3, 5.4, 5.5, 5.6)
    return lo + hi


def config2(seed: int = 101, n_mcs: int = 20000) -> Config:
    """BASELINE.json configs[1]: L=400, r sweep, 20000 MCS (last 10000 averaged)."""
    rs = config2_rs()
    return Config("C2_L400_rsweep", 400, rs, tuple(seed for _ in rs), n_mcs,
                  note="one lattice per r, same seed")


def config3(r: float = 3.7443, n_mcs: int = 100000) -> Config:
    """BASELINE.json configs[2]: L=2048 critical decay, 16 seeds (1..16)."""
    return Config("C3_L2048_decay", 2048, tuple(r for _ in range(16)), tuple(range(1, 17)), n_mcs)


def config4(n_mcs: int = 10000) -> Config:
    """BASELINE.json configs[3]: 64 lattices L=512, r_k = 3.70 + (0.1*k)/63, seeds 1000+k."""
    rs = tuple(3.70 + (0.1 * k) / 63.0 for k in range(64))
    return Config("C4_ens64_L512", 512, rs, tuple(1000 + k for k in range(64)), n_mcs)


def config5(n_mcs: int = 1000, L: int = 16384) -> Config:
    """BASELINE.json configs[4]: the throughput lattice, L=16384, r=3.8, seed 1."""
    return Config("C5_L16384", L, (3.8,), (1,), n_mcs)


ALL = {"c1": config1, "c2": config2, "c3": config3, "c4": config4, "c5": config5}


# --------------------------------------------------------------------------
# Arbitrary seeded lattices (numpy generator -- not the method's Philox init)
# --------------------------------------------------------------------------
def random_lattice(L: int, p: float, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return (rng.random((L, L)) < p).astype(np.uint8)


def blobs_lattice(L: int, seed: int, n_blobs: int = 12) -> np.ndarray:
    """Compact cooperator clusters in a defector sea (cooperators
    survive by forming compact clusters) -- exercises interfaces and bulk."""
    rng = np.random.default_rng(seed)
    lat = np.zeros((L, L), dtype=np.uint8)
    ii, jj = np.meshgrid(np.arange(L), np.arange(L), indexing="ij")
    for _ in range(n_blobs):
        ci, cj = rng.integers(0, L, size=2)
        rad = rng.integers(2, max(3, L // 6))
        di = np.minimum((ii - ci) % L, (ci - ii) % L)
        dj = np.minimum((jj - cj) % L, (cj - jj) % L)
        lat[(di * di + dj * dj) <= rad * rad] = 1
    return lat


def stripes_lattice(L: int, width: int = 5, vertical: bool = True) -> np.ndarray:
    a = (np.arange(L) // width) % 2
    lat = np.broadcast_to(a[None, :] if vertical else a[:, None], (L, L))
    return np.ascontiguousarray(lat, dtype=np.uint8)


def checkerboard_lattice(L: int) -> np.ndarray:
    ii, jj = np.meshgrid(np.arange(L), np.arange(L), indexing="ij")
    return ((ii + jj) % 2).astype(np.uint8)
