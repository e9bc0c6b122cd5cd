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


def test_both_arms_describe_the_same_config():
    sys.path.insert(0, ROOT)
    import bench
    import workloads as W
    cfg = W.get("cfg3")
    a, b = bench.config_dict(cfg, 1), bench.config_dict(cfg, 1)
    assert a == b and a["workload"] == cfg.name and "model" not in a
    src = open(os.path.join(ROOT, "bench.py")).read()
    assert src.count('"config": config_dict(') == 2        # ours and the reference arm


def test_traffic_lookup_follows_the_kernel_sha(tmp_path, monkeypatch):
    """roofline.traffic comes from profiles/traffic.json only while the sweep-kernel sources are the
    ones the ncu capture was taken at; otherwise null (never a stale constant)."""
    sys.path.insert(0, ROOT)
    import bench
    tab = json.load(open(bench.TRAFFIC_JSON))
    assert set(tab["workloads"]) >= {"cfg3_96c_periodic_f64", "cfg4_72c_bloch_c128",
                                     "cfg5_slab_128x128x192_f64"}
    got = bench.ncu_traffic("cfg3_96c_periodic_f64")
    if tab["kernel_sha"] == bench.kernel_sha():
        assert got == tab["workloads"]["cfg3_96c_periodic_f64"]["dram_bytes"]
        import workloads as W
        assert 1.0 <= got / W.get("cfg3").min_bytes < 1.1
    else:
        assert got is None
    stale = dict(tab, kernel_sha="0" * 16)
    f = tmp_path / "traffic.json"
    f.write_text(json.dumps(stale))
    monkeypatch.setattr(bench, "TRAFFIC_JSON", str(f))
    assert bench.ncu_traffic("cfg3_96c_periodic_f64") is None
    assert bench.ncu_traffic("no_such_workload") is None
