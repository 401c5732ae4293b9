"""N > 1 path of bench.py on CPU: two gloo ranks, replicas only.  What is shared between
ranks is one MAX-reduction of the timing scalar and rank 0 printing the aggregate; there is no data-path collective."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = 100.0 + 50.0 * rank                       # rank 1 is the slow replica
tmax = bench.reduce_max(ms, world, torch.device("cpu"))
val = bench.aggregate_value(ntraj=3, world=world, ms_per_step=tmax)
if rank == 0:
    print(json.dumps({{"tmax": tmax, "value": val, "world": world}}))
dist.destroy_process_group()
"""


def test_two_rank_timing_reduction_and_aggregate(tmp_path):
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    d = json.loads(outs[0][0].strip().splitlines()[-1])
    assert d["world"] == 2 and d["tmax"] == 150.0                       # max over ranks, not the mean
    assert abs(d["value"] - 8 * 3 * 2 / 0.150) < 1e-9                   # whole-job sigma-vectors/s


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
