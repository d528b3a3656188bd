"""bench.py's N > 1 logic on CPU: the path does not shard (replicas only), so
every rank times its own replica and rank 0 reports N * particles / max-over-ranks time. This test
runs that reduction with world size 2 on the gloo backend, and the reference arm's rank gating."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_replica_aggregation_gloo_world2(tmp_path):
    script = tmp_path / "agg.py"
    script.write_text(textwrap.dedent(f"""
        import os, sys, json
        sys.path.insert(0, {ROOT!r})
        import torch, torch.distributed as dist
        import bench
        dist.init_process_group("gloo")
        rank, world = dist.get_rank(), dist.get_world_size()
        ms = [10.0, 14.0][rank]                      # this rank's summed step times
        total, e2e = bench.max_over_ranks(ms, ms * 2, world, torch.device("cpu"))
        value = bench.whole_job_value(world, 1000, 5, total)
        if rank == 0:
            print(json.dumps({{"total": total, "e2e": e2e, "value": value}}))
        dist.destroy_process_group()
    """))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29533")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29533", str(script)],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    import json
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    r = json.loads(line)
    assert r["total"] == 14.0 and r["e2e"] == 28.0               # max over ranks
    assert abs(r["value"] - 2 * 1000 * 5 / 14e-3) < 1e-6         # all ranks' particles / slowest rank


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--workload", "cfg1_open512", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""      # other ranks exit 0 without work
    env["RANK"] = "0"
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--workload", "cfg1_open512", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, env=env, timeout=300)
    import json
    r = json.loads(out.stdout.strip().splitlines()[-1])
    assert r["impl"] == "reference" and r["cpu_baseline"]["kind"] == "oracle" and r["value"] > 0
    assert r["e2e"]["h2d_bytes_per_step"] == 0
