"""The N > 1 path of bench.py on CPU: two processes over gloo (127.0.0.1).

The hot path does not shard at BASELINE.json's sizes (replicas only), so
the only cross-rank logic is bench.py's: barrier, max-over-ranks of the device time, whole-job
value = plans of all ranks / that time, and rank 0 alone printing.  The reference arm under
torchrun: rank 0 alone runs, the other ranks exit without work.
"""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
dist.barrier()
local = 0.100 + 0.050 * rank                      # rank 1 is the slow replica
mx = bench.reduce_max(local, world, device="cpu")
val = bench.job_seconds_per_plan(mx, steps=5, world=world)
dist.barrier()
json.dump({{"rank": rank, "max": mx, "value": val}}, open(os.path.join({out!r}, f"r{{rank}}.json"), "w"))
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_max_over_ranks_and_whole_job_value(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT, out=str(tmp_path)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    res = [json.load(open(tmp_path / f"r{i}.json")) for i in range(2)]
    for x in res:
        assert abs(x["max"] - 0.150) < 1e-12                 # every rank sees the slowest rank's time
        assert abs(x["value"] - 0.150 / (5 * 2)) < 1e-12     # 2 replicas x 5 plans in 0.150 s


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_max(0.25, 1) == 0.25
    assert bench.job_seconds_per_plan(1.0, 5, 1) == 0.2


def test_reference_arm_runs_on_rank0_only(tmp_path):
    """`bench.py --impl reference` with RANK=1: exits 0 without output and without touching the oracle."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=120, env=env)
    assert r.returncode == 0 and r.stdout.strip() == ""


@pytest.mark.slow
def test_reference_arm_prints_contract_line():
    """Rank 0 of the reference arm on the small config: one JSON line with the contract's keys."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "cfg0",
                        "--steps", "1", "--warmup", "0", "--ref-apertures", "2"], capture_output=True, text=True,
                       timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "s" and line["higher_is_better"] is False
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] == 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["value"] == line["value"]
