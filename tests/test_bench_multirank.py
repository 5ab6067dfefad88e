"""Host logic of the N > 1 path of bench.py on CPU: world_size-2 gloo process group (the path does not
shard — "replicas only", DESIGN.md §8 — so the only collective is the max-over-ranks of the step time),
and the reference arm's rank gating under torchrun-style environments."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
rank = int(os.environ["RANK"])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%%s" %% os.environ["MASTER_PORT"],
                        rank=rank, world_size=2)
ms = bench.max_over_ranks(3.0 + 2.0 * rank, dist, torch.device("cpu"))       # rank 0: 3 ms, rank 1: 5 ms
val = bench.aggregate_value(1000, 2, ms)
print("RESULT %%d %%.6f %%.3f" %% (rank, ms, val), flush=True)
dist.destroy_process_group()
'''


def test_max_over_ranks_and_aggregate_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    port = str(29500 + os.getpid() % 2000)
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=port)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    for r, out in enumerate(outs):
        line = [l for l in out.splitlines() if l.startswith("RESULT")][0].split()
        assert int(line[1]) == r
        assert float(line[2]) == 5.0                       # the slower rank decides
        assert float(line[3]) == pytest.approx(2 * 1000 / 5e-3)   # both replicas' updates / max time


def test_single_process_helpers():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(1.25, None, None) == 1.25
    assert bench.aggregate_value(640, 1, 2.0) == pytest.approx(320000.0)


def test_reference_arm_rank_gating():
    """Under torchrun only rank 0 runs and prints the reference line; other ranks exit 0 without work."""
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "config1",
           "--nvis", "4096", "--steps", "1", "--warmup", "0", "--gpus", "2"]
    out1 = subprocess.run(cmd, env=dict(os.environ, RANK="1", WORLD_SIZE="2"), capture_output=True, text=True, timeout=300)
    assert out1.returncode == 0 and out1.stdout.strip() == ""
    out0 = subprocess.run(cmd, env=dict(os.environ, RANK="0", WORLD_SIZE="2"), capture_output=True, text=True, timeout=300)
    assert out0.returncode == 0, out0.stderr
    d = json.loads(out0.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["config"]["workload"] == "config1"
