"""N>1 path of bench.py on CPU (gloo, world_size 2): replicas only -- each rank times its own solves, the job
time is the max over ranks, the value is all ranks' solves over that time; the reference arm prints on rank 0
only."""
import json
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys, json
    sys.path.insert(0, %r)
    import torch, torch.distributed as dist
    import bench
    dist.init_process_group(backend="gloo")
    rank = dist.get_rank()
    ms = 10.0 if rank == 0 else 25.0          # rank 1 is the slow replica
    mx = bench.max_over_ranks(torch, dist, ms)
    v = bench.job_value(dist.get_world_size(), 4, 5, mx)
    if rank == 0:
        print(json.dumps({"max_ms": mx, "value": v}))
    dist.barrier()
    dist.destroy_process_group()
""" % ROOT)


def test_max_over_ranks_and_job_value_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29611", str(script)],
                         capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    r = json.loads(line)
    assert r["max_ms"] == 25.0
    assert abs(r["value"] - 2 * 4 * 5 / 0.025) < 1e-9


def test_reference_arm_rank0_only_and_contract_keys():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                          "--config", "cfg0"], capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2", "--warmup", "1",
                          "--config", "cfg0"], capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    r = json.loads(out.stdout.strip().splitlines()[-1])
    assert r["impl"] == "reference" and r["unit"] == "solves/s" and r["value"] > 0
    assert r["cpu_baseline"]["kind"] == "oracle" and r["cpu_baseline"]["cores"] >= 1
    assert r["e2e"]["h2d_bytes_per_step"] == 0 and r["e2e"]["value"] == r["value"]
