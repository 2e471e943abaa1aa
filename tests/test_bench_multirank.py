"""Host-side logic of bench.py's N > 1 path (replicas only), covered on
CPU with world_size 2 over gloo: max-over-ranks timing, whole-job value, per-rank seeds, and the
reference arm's "rank 0 alone prints" rule."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
ms = bench.max_over_ranks(10.0 + 5.0 * rank, torch.device("cpu"), world)     # rank 1 is the slow one
val = bench.whole_job_value(1000.0, world, ms * 1e-3)
out = dict(rank=rank, ms=ms, value=val, seed=bench.replica_seed(7, rank))
dist.barrier()
print("RESULT " + json.dumps(out), flush=True)
dist.destroy_process_group()
"""


def test_max_over_ranks_and_whole_job_value_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = 29500 + (os.getpid() % 2000)
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port),
                   LOCAL_RANK=str(rank))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=300)
        assert p.returncode == 0, e
        line = [l for l in o.splitlines() if l.startswith("RESULT ")][0]
        outs.append(json.loads(line[7:]))
    outs.sort(key=lambda d: d["rank"])
    assert [d["ms"] for d in outs] == [15.0, 15.0]                       # MAX over ranks on both
    assert all(abs(d["value"] - 2 * 1000.0 / 15e-3) < 1e-6 for d in outs)  # whole job = sum of the replicas' rates
    assert [d["seed"] for d in outs] == [7, 8]


def test_reference_arm_only_rank0_prints():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_line_shape():
    env = dict(os.environ)
    env.pop("RANK", None)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "0", "--ref-samples", "4", "--ref-walks", "2", "--faces", "20000", "--components", "5",
                        "--samples", "200", "--candidates", "5000", "--walks", "64", "--no-cache"],
                       env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    d = json.loads(r.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["metric"] == "walk_steps_per_s" and d["vs_baseline"] is None
    assert d["config"]["workload"].startswith("configs[3]")
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"] and d["gpu_launches"] == 0
