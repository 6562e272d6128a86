"""Host-side logic of bench.py's N > 1 path (replicas only: the hot path does not shard),
exercised with two CPU processes over gloo: every rank must see the slowest rank's time, the whole-job value is
the replicas' bytes over that time, and only rank 0 of the reference arm does any work."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["SLDG_ROOT"])
import torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, device="cpu")
val = bench.replicas_value(8.0e9, ms, world)
dist.barrier()
dist.destroy_process_group()
print(json.dumps({"rank": rank, "ms": ms, "value": val}))
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_ranks_agree_on_the_slowest_time_and_the_aggregate_value():
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port),
                   SLDG_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        outs.append(json.loads(out.strip().splitlines()[-1]))
    assert [o["ms"] for o in outs] == [15.0, 15.0]
    expect = 2 * 8.0e9 / 15.0e-3 / 1e9
    assert all(abs(o["value"] - expect) < 1e-9 * expect for o in outs)


def test_reference_arm_runs_on_rank_0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=240)
    assert r.returncode == 0 and r.stdout.strip() == ""
