"""Host-side logic of bench.py's N > 1 path, on CPU with the gloo backend (world_size 2).

The hot path does not shard (replicas only), so the only collective is the
max-over-ranks reduction of the timings, and the reference arm must run on rank 0 alone."""
import json
import os
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]
sys.path.insert(0, str(ROOT))

torch = pytest.importorskip("torch")


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = [10.0 + rank, 5.0 - rank]          # rank 1 is slower on the first, faster on the second
    got = bench.max_over_ranks(mine, world)
    value = bench.job_value(world, 3, 1000.0, got[0])
    dist.barrier()
    dist.destroy_process_group()
    Path(out, f"r{rank}.json").write_text(json.dumps({"got": got, "value": value}))


def test_max_over_ranks_and_job_value_world2(tmp_path):
    import torch.multiprocessing as mp
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    for rank in range(2):
        r = json.loads((tmp_path / f"r{rank}.json").read_text())
        assert r["got"] == [11.0, 5.0]                       # max over ranks, same on every rank
        assert r["value"] == pytest.approx(2 * 3 * 1000.0 / 11e-3)


def test_single_rank_is_identity():
    import bench
    assert bench.max_over_ranks([1.5, 2.5], 1) == [1.5, 2.5]
    assert bench.job_value(1, 2, 100.0, 1000.0) == pytest.approx(200.0)


def test_reference_arm_under_torchrun_prints_one_line(tmp_path):
    """torchrun with 2 ranks: rank 0 times the oracle and prints the JSON line, rank 1 exits 0."""
    port = 31500 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(ROOT / "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "2", "--warmup", "1", "--L", "256"]
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [ln for ln in p.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["steps"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
