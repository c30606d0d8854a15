"""Host-side logic of bench.py on CPU: the N>1 aggregation (max time over ranks, units summed) over a world_size-2
gloo group, the bounded oracle sample of the reference arm, and the reference arm's JSON line."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r took (2 + r) ms for (100 + r) units: whole job = max time, summed units
    ms, units = bench.aggregate_over_ranks(2.0 + rank, 100.0 + rank, dist)
    with open(out % rank, "w") as f:
        json.dump({"ms": ms, "units": units}, f)
    dist.destroy_process_group()


def test_aggregate_over_ranks_gloo_world2(tmp_path):
    torch = pytest.importorskip("torch")
    import torch.multiprocessing as mp
    out = str(tmp_path / "r%d.json")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    for r in range(2):
        got = json.load(open(out % r))
        assert got == {"ms": 3.0, "units": 201.0}


def test_aggregate_single_process_is_identity():
    assert bench.aggregate_over_ranks(1.5, 7.0, None) == (1.5, 7.0)


def test_reference_sample_is_bounded_power_of_two():
    for steps, warmup in [(1, 0), (10, 3), (100, 50)]:
        Ls = bench.reference_sample_L(16384, steps, warmup)
        assert 64 <= Ls <= 16384 and (Ls & (Ls - 1)) == 0
        # the whole run fits the budget at the assumed oracle speed
        assert (steps + warmup) * Ls * Ls * 160e-9 <= 150.0 or Ls == 64
    assert bench.reference_sample_L(64, 1, 0) == 64


def test_reference_arm_prints_one_json_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--L", "128",
                        "--steps", "2", "--warmup", "3"], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr
    lines = [ln for ln in r.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "ns" and d["higher_is_better"] is False
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["value"] > 0


def test_reference_arm_nonzero_rank_is_silent():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--L", "128", "--steps", "1"], capture_output=True, text=True, timeout=120, env=env)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_bench_percolation_thresholds_are_the_stored_golden_integers():
    """bench.py passes BASELINE.json configs[3]'s bond thresholds to sw_set_threshold as integers; they are the values of
    tests/golden/thresholds.txt (pinned there to the closed forms), not something the bench computes."""
    from conftest import read_golden
    g = read_golden("thresholds.txt")
    assert bench.PERC_THRESHOLD == {0.3: int(g["perc_0.3"]), 0.5: int(g["perc_0.5"]), 0.7: int(g["perc_0.7"])}
