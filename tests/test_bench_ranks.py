"""The N > 1 path of bench.py is "replicas only": no data-path collective, the job's time is the
max over ranks, the value the sum of the replicas' work.  Covered here with a world_size-2 gloo group on the CPU."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
ms = bench.max_over_ranks(10.0 if dist.get_rank() == 0 else 25.0)       # rank 1 is the slow replica
val = bench.aggregate_value(1.0e9, ms, dist.get_world_size())
dist.barrier()
if dist.get_rank() == 0:
    print("RESULT", ms, val)
dist.destroy_process_group()
"""


def test_replicas_take_the_max_time_and_sum_the_work(tmp_path):
    pytest.importorskip("torch")
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT, port=29731))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=240) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    line = [l for l in outs[0][0].splitlines() if l.startswith("RESULT")][0].split()
    assert float(line[1]) == 25.0                                   # max over ranks
    assert abs(float(line[2]) - 2 * 1.0e9 / 25.0e-3 / 1e9) < 1e-9    # two replicas' bytes over the slowest time


def test_single_process_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.aggregate_value(2.0e9, 1.0, 1) == 2000.0


def test_reference_arm_prints_only_on_rank0():
    """bench.py --impl reference under torchrun: rank 0 alone runs and prints, the other ranks exit 0 without work."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "1"], capture_output=True, text=True, env=env, timeout=240)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="2", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "1"], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["n_gpus"] == 2
