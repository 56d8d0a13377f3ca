"""N > 1 path of bench.py on CPU (gloo, world_size 2). The hot path does not shard ("replicas only",
DESIGN.md section 8): the only cross-rank logic is the max-over-ranks of the device times and the whole-job
aggregate, plus `--impl reference` running on rank 0 alone."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
local_ms = 100.0 * (rank + 1)                       # rank 1 is the slow one
value, ms_step = bench.aggregate_throughput(1000, 10, local_ms, world, device="cpu")
t = bench.max_over_ranks(0.5 + rank, device="cpu")
dist.barrier()
print(json.dumps({{"rank": rank, "value": value, "ms_step": ms_step, "tmax": t}}))
dist.destroy_process_group()
"""


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_max_over_ranks_and_aggregate_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, text=True))
    outs = [json.loads(p.communicate(timeout=120)[0].strip().splitlines()[-1]) for p in procs]
    assert all(p.returncode == 0 for p in procs)
    for o in outs:
        # slowest rank: 200 ms for 10 steps; whole job = 2 ranks x 1000 units x 10 steps / 0.2 s
        assert abs(o["ms_step"] - 20.0) < 1e-9 and abs(o["value"] - 2 * 1000 * 10 / 0.2) < 1e-6
        assert o["tmax"] == 1.5


def test_single_process_aggregate_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    value, ms_step = bench.aggregate_throughput(192000, 50, 545.0, 1, device="cpu")
    assert abs(ms_step - 10.9) < 1e-12 and abs(value - 192000 * 50 / 0.545) < 1e-3


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--config", "1"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""          # other ranks exit 0 without work
    env["RANK"] = "0"; env["LOCAL_RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--config", "1", "--ref-atoms", "96"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "atom-steps/s"
