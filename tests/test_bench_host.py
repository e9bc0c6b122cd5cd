"""Host-side logic of bench.py that needs no GPU: the N>1 aggregation over gloo (world size 2)
and the --impl reference arm (the CPU oracle as its own bench line)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_aggregate_two_ranks_gloo():
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29731",
           os.path.join(ROOT, "tests", "_gloo_worker.py")]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    line = [l for l in res.stdout.splitlines() if l.startswith("{")][-1]
    out = json.loads(line)
    # slowest rank took 2 ms; two replicas of 1e9 units each -> 2e9 units / 2 ms = 1000 G/s
    assert out["world"] == 2 and out["ms"] == 2.0
    assert abs(out["value"] - 1000.0) < 1e-9


def test_aggregate_single_rank_is_plain_rate():
    sys.path.insert(0, ROOT)
    import bench
    value, t = bench.aggregate(0.5, 2e9, 1, lambda x: x)
    assert t == 0.5 and abs(value - 4000.0) < 1e-9


def test_reference_arm_prints_contract_line():
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload",
           "cfg1", "--steps", "2", "--warmup", "1"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    d = json.loads(res.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["unit"] == "Gpoint.band/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
    assert d["higher_is_better"] is True and d["vs_baseline"] is None
