"""Host-side logic of the N > 1 path ("replicas only"): rank discovery, barrier and the
max-over-ranks reduction bench.py uses, exercised with world_size 2 over gloo on the CPU; plus the
--impl reference arm (CPU oracle) end to end."""
import json
import os
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group(backend="gloo")
rank = dist.get_rank()
bench.barrier()
local_ms = 10.0 + 5.0 * rank                  # rank 1 is the slow one
worst = bench.reduce_max(local_ms)            # CPU tensor over gloo
steps = 7
value = dist.get_world_size() * steps / (worst * 1e-3)   # whole-job solves/s: all ranks' solves / slowest rank's time
bench.barrier()
if rank == 0:
    print(json.dumps({{"worst": worst, "value": value, "world": dist.get_world_size()}}))
dist.destroy_process_group()
"""


def test_replica_aggregation_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=str(ROOT)))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run(
        [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
         "--master-port", "29533", str(script)], capture_output=True, text=True, timeout=240, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["world"] == 2 and d["worst"] == 15.0
    assert d["value"] == pytest.approx(2 * 7 / 15e-3)


def test_reference_arm_prints_contract_line():
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--config", "c0", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads(out.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["metric"] == "poisson_solves_per_sec" and d["unit"] == "solves/s"
    assert d["value"] > 0 and d["higher_is_better"] is True and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--config", "c0", "--gpus", "2"],
                         capture_output=True, text=True, timeout=120, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""
