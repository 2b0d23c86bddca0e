"""Multi-rank host logic of bench.py on CPU (gloo, world size 2): replicas only.

The data path has no collective; what a multi-rank run shares is the MAX over the ranks' timed regions and the
whole-job aggregate printed by rank 0, and `--impl reference` runs on rank 0 alone.  No GPU, no CUDA extension.
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
dist.init_process_group("gloo", rank=rank, world_size=world)
# every rank 'timed' a different region: the job is as slow as its slowest replica
local = [10.0 + 5.0 * rank, 100.0 - 20.0 * rank]
mx = bench.replica_max_times(local, world, "cpu")
dist.barrier()
out = {{"rank": rank, "max": mx, "value": bench.aggregate_value(1000, 50, world, mx[0])}}
print("RESULT " + json.dumps(out), flush=True)
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _spawn(world, code):
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", code], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True, cwd=ROOT))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=240)
        assert p.returncode == 0, e[-2000:]
        outs.append(o)
    return outs


@pytest.mark.timeout(300)
def test_two_replicas_max_over_ranks_and_aggregate():
    outs = _spawn(2, WORKER.format(root=ROOT))
    res = sorted((json.loads(l[7:]) for o in outs for l in o.splitlines() if l.startswith("RESULT ")),
                 key=lambda d: d["rank"])
    assert [d["rank"] for d in res] == [0, 1]
    for d in res:
        assert d["max"] == [15.0, 100.0]                       # MAX over ranks, per timed region
        assert d["value"] == pytest.approx(2 * 1000 * 50 / 15.0e-3)   # all ranks' units / slowest rank's time


@pytest.mark.timeout(300)
def test_reference_arm_runs_on_rank0_only():
    """`--impl reference` under torchrun: rank 0 times the oracle and prints the line, the others exit 0 silently."""
    outs = []
    for r in (0, 1):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(_free_port()))
        p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                            "--config", "1", "--steps", "2", "--warmup", "1"], env=env, capture_output=True,
                           text=True, cwd=ROOT, timeout=280)
        assert p.returncode == 0, p.stderr[-2000:]
        outs.append(p.stdout)
    lines = [l for l in outs[0].splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["n_gpus"] == 2
    assert outs[1].strip() == ""
