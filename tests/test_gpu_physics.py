"""Statistics of the sublattice schedule on the GPU against the random-sequential oracle (``-m gpu``).

BASELINE.json configs[1] (L=400, K=0.5, 20000 MCS, last 10000 averaged).  The
random-sequential numbers were written by ``tests/golden/make_rs_stats.py`` (oracle only, seeds
201/202); the GPU runs the 16-sublattice schedule with seeds 101-104.  The two are different
stochastic processes, so only statistics can agree:
|mean_GPU - mean_RS| <= 3.5 sqrt(sigma_GPU^2 + sigma_RS^2) + 5e-4, sigma from batch means and
the scatter between seeds.  PERM (every site exactly once per MCS) is expected to FAIL this:
the test pins that finding too, so a silent change of the default order mode shows up."""
import collections
import json
import math
from pathlib import Path

import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import paper_1704_08098_b200 as pgg  # noqa: E402
from paper_1704_08098_b200 import physics  # noqa: E402

RS = json.loads((Path(__file__).resolve().parent / "golden" / "C2_rs_stats.json").read_text())


def rs_table():
    by = collections.defaultdict(list)
    for row in RS["rows"]:
        by[row["r"]].append(row)
    out = {}
    for r, rows in by.items():
        mean = sum(q["mean"] for q in rows) / len(rows)
        within = math.sqrt(sum(q["stderr"] ** 2 for q in rows)) / len(rows)
        between = (max(q["mean"] for q in rows) - min(q["mean"] for q in rows)) / 2 if len(rows) > 1 else 0.0
        out[r] = (mean, max(within, between))
    return out


@pytest.fixture(scope="module")
def gpu_tables():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (there is no CPU fallback)")
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)
    rs = sorted(rs_table())
    args = dict(L=RS["L"], n_mcs=RS["n_mcs"], K=RS["K"], rho0=RS["rho0"])
    return (physics.stationary(rs, [101, 102, 103, 104], order=pgg.ORDER_IID, **args),
            physics.stationary(rs, [101, 102, 103, 104], order=pgg.ORDER_PERM, **args))


def n_sigma(g, ref):
    return (g["mean"] - ref[0]) / (math.sqrt(g["stderr"] ** 2 + ref[1] ** 2) + 1e-12)


def test_iid_schedule_matches_random_sequential(gpu_tables):
    iid, _ = gpu_tables
    ref = rs_table()
    for r, g in iid.items():
        tol = 3.5 * math.sqrt(g["stderr"] ** 2 + ref[r][1] ** 2) + 5e-4
        assert abs(g["mean"] - ref[r][0]) <= tol, f"r={r}: GPU IID {g['mean']:.4f} vs RS {ref[r][0]:.4f} (tol {tol:.4f})"


def test_extinction_and_full_cooperation_limits(gpu_tables):
    """Below r_c = 3.7443(4) cooperators die out; the upper transition to full
    cooperation lies between 5.5 and 5.6 for both schedules."""
    iid, _ = gpu_tables
    for r in (3.6, 3.65, 3.7):
        assert iid[r]["mean"] == 0.0
    assert iid[3.75]["mean"] > 0.02          # finite-size L=400: still alive just above r_c
    assert 0.99 < iid[5.5]["mean"] < 1.0 and iid[5.6]["mean"] > 0.9999
    means = [iid[r]["mean"] for r in sorted(iid)]
    assert all(b >= a - 1e-3 for a, b in zip(means, means[1:])), "rho_C(r) must be non-decreasing"


def test_perm_order_is_biased(gpu_tables):
    """The literal "each class exactly once per MCS" reading does not reproduce random-sequential
    statistics: rho_C is too high by tens of sigma for 3.75 <= r <= 4."""
    _, perm = gpu_tables
    ref = rs_table()
    for r in (3.8, 3.9, 4.0):
        assert n_sigma(perm[r], ref[r]) > 10.0


def test_critical_decay_brackets_the_threshold():
    """BASELINE.json configs[2] at its size and length (L = 2048, 16 seeds, 10^5 MCS; bit-packed, so the
    run takes about a minute): on either side of the threshold r_c = 3.7445(1) (
    the paper: 3.7443(4)) the local decay exponent delta_eff(t) = -ln[rho(t)/rho(t/8)]/ln 8
    bends the way directed percolation says it must: below r_c it keeps growing past the
    DP value 0.4505 (the density dies exponentially), above r_c it falls back towards 0 (the density
    saturates).  The decay from a random start is not a clean power law before t ~ 10^4 (S20), so only the
    last decade is used."""
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)
    seeds = list(range(1, 17))

    def d_eff(r):
        rows = {q["t"]: q for q in physics.decay(r, seeds, L=2048, n_mcs=100000, fmt=pgg.FMT_BITS)}
        ts = sorted(rows)
        late = [rows[t] for t in ts if t >= 30000 and "delta_eff" in rows[t]]
        return rows, late

    sub_rows, sub = d_eff(3.7440)
    sup_rows, sup = d_eff(3.7450)
    # sub-critical: delta_eff passes the DP value and keeps rising (or the seeds die out altogether)
    dead = sub_rows[100000]["alive"] == 0
    assert dead or sub[-1]["delta_eff"] > 0.4505 + 3 * sub[-1]["delta_err"], sub[-1]
    assert dead or sub[-1]["delta_eff"] > sub[0]["delta_eff"]
    # super-critical: every seed alive, delta_eff stays below the DP value and has stopped growing
    assert sup_rows[100000]["alive"] == len(seeds)
    assert sup[-1]["delta_eff"] < 0.4505 - 3 * sup[-1]["delta_err"], sup[-1]
    assert sup[-1]["delta_eff"] < max(q["delta_eff"] for q in sup) + 1e-12
    assert sup_rows[100000]["rho"] > 2 * sub_rows[100000]["rho"]
