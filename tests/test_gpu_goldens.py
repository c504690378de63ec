"""Full-length parity on BASELINE.json configs 2-5 against stored oracle results (``-m gpu``).

``tests/golden/make_goldens.py`` (which calls only ``oracle/``) ran every lattice of a
config on the CPU and stored count0, the SHA-256 of the whole cooperator-count trace,
counts at log-spaced MCS and the SHA-256 of the lattice at snapshot times.  Here the same
configs run through the C ABI on the GPU, in the ensemble launch the library uses for
them, and every stored value must be reproduced bit for bit.  No GPU-produced state is
ever fed to the oracle."""
import hashlib
import json
from pathlib import Path

import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import paper_1704_08098_b200 as pgg  # noqa: E402

GOLDEN = Path(__file__).resolve().parent / "golden"
FILES = sorted(GOLDEN.glob("C[2-5]_*_mcs*.json"))


def unpack(words, L):
    bits = (words.view(np.uint32)[..., None] >> np.arange(32, dtype=np.uint32)) & 1
    return bits.reshape(words.shape[:-1] + (L,)).astype(np.uint8)


def lattice_sha(d_lat, fmt, L):
    a = d_lat.cpu().numpy()
    if fmt == pgg.FMT_BITS:
        a = unpack(a, L)
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


@pytest.mark.parametrize("fmt", [pgg.FMT_U8, pgg.FMT_BITS])
@pytest.mark.parametrize("path", FILES, ids=[f.stem for f in FILES])
def test_config_reproduces_stored_oracle_run(path, fmt):
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (there is no CPU fallback)")
    g = json.loads(path.read_text())
    L, K, rho0, n_mcs = g["L"], g["K"], g["rho0"], g["n_mcs"]
    if fmt == pgg.FMT_BITS and L % 32:
        pytest.skip("bits layout needs L % 32 == 0")
    members = g["members"]
    B = len(members)
    rs = [float.fromhex(m["r_hex"]) for m in members]
    seeds = [m["seed"] for m in members]
    pgg.pgg_set_variant(pgg.VARIANT_AUTO)
    shape = (B, L, L) if fmt == pgg.FMT_U8 else (B, L, L // 32)
    d = torch.empty(shape, dtype=torch.uint8 if fmt == pgg.FMT_U8 else torch.int32, device="cuda")
    cnt0 = torch.zeros(B, dtype=torch.int64, device="cuda")
    traces, t = [], 0
    for stop in sorted(set(g["snapshots"] + [n_mcs])):
        n = stop - t
        cnt = torch.zeros((B, n), dtype=torch.int64, device="cuda")
        # first segment initialises (rho0 in [0,1]); later ones continue (rho0 < 0)
        pgg.pgg_run_ensemble(d, fmt, B, L, rs, K, seeds, pgg.ORDER_IID, rho0 if t == 0 else -1.0, t, n, cnt)
        if t == 0:
            # count0 from a separate init (the ensemble call above has already swept)
            d0 = torch.empty(shape[1:], dtype=d.dtype, device="cuda")
            for b in range(B):
                pgg.pgg_init_lattice(d0, fmt, L, rho0, seeds[b])
                pgg.pgg_density(d0, fmt, L, cnt0[b:b + 1])
        torch.cuda.synchronize()
        traces.append(cnt.cpu().numpy().astype("<u8"))
        t = stop
        if stop in g["snapshots"]:
            for b, m in enumerate(members):
                assert lattice_sha(d[b], fmt, L) == m["snap_sha256"][str(stop)], \
                    f"{g['config']} member {b} (r={m['r']}, seed={m['seed']}): lattice differs at MCS {stop}"
    trace = np.concatenate(traces, axis=1)
    for b, m in enumerate(members):
        assert int(cnt0[b].item()) == m["count0"]
        for s, v in m["samples"].items():
            assert int(trace[b, int(s) - 1]) == v, f"{g['config']} member {b}: count after MCS {s}"
        assert hashlib.sha256(np.ascontiguousarray(trace[b]).tobytes()).hexdigest() == m["trace_sha256"], \
            f"{g['config']} member {b}: rho_C trace differs"


def test_golden_files_exist():
    names = {f.name.split("_")[0] for f in FILES}
    assert {"C2", "C3", "C4", "C5"} <= names, f"missing golden files, have {sorted(names)}"
