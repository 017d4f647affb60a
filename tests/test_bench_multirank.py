"""The N > 1 path of bench.py ("replicas only") on CPU: two gloo ranks, the only cross-rank
operation is the MAX of the per-rank timings; the reported value is all ranks' particle-steps over that time."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_max_over_ranks_and_rate_world2_gloo(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(textwrap.dedent(f"""
        import os, sys, json
        sys.path.insert(0, {ROOT!r})
        import torch.distributed as dist
        import bench
        dist.init_process_group("gloo")
        rank, world = dist.get_rank(), dist.get_world_size()
        ms, e2e = (10.0, 2.0) if rank == 0 else (12.5, 1.0)      # rank 1 is slower on the device, rank 0 end to end
        out = bench.max_over_ranks([ms, e2e], world, "cpu")
        rate = bench.whole_job_rate(1000, 50, world, out[0] * 1e-3)
        if rank == 0:
            print(json.dumps({{"out": out, "rate": rate}}))
        dist.destroy_process_group()
    """))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29641")
    res = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29641", str(script)],
                         capture_output=True, text=True, env=env, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    import json
    line = [l for l in res.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["out"] == [12.5, 2.0]
    assert abs(d["rate"] - 2 * 1000 * 50 / 12.5e-3) < 1e-6


def test_reference_arm_prints_one_json_line():
    """bench.py --impl reference: the oracle on a bounded sample, same keys as our arm."""
    import json
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2",
                          "--warmup", "1", "--workload", "0"], capture_output=True, text=True, timeout=600)
    assert res.returncode == 0, res.stderr[-2000:]
    d = json.loads(res.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["unit"] == "particle-steps/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["vs_baseline"] is None and d["higher_is_better"] is True


def test_single_rank_helpers():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.0, 2.0], 1, "cpu") == [1.0, 2.0]
    assert bench.whole_job_rate(10, 5, 1, 0.5) == 100.0
    assert 6 <= bench.oracle_sample_edge(1e3) <= bench.oracle_sample_edge(1e9) <= 40
    assert bench.algorithmic_bytes("k_force", 10, 49.0, 25.0) == 10 * (48 + 50)
    assert bench.algorithmic_ops("k_force", 10, 49.0, 25.0) == 10 * 48 * 25.0
