"""The only N>1 logic of this repo ("replicas only"): max-over-ranks timing and the whole-job
aggregate in bench.py.  Run with two gloo ranks on the CPU."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
rank, ws = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=ws)
ms, e2e = bench.max_over_ranks([10.0 + 5.0 * rank, 100.0 - 7.0 * rank], ws)
ws_, rank_, lr_ = bench._dist()
assert (ws_, rank_) == (ws, rank)
if rank == 0:
    print(json.dumps({"ms": ms, "e2e": e2e, "value": bench.aggregate_value(1000, 4, ms, ws)}))
dist.barrier()
dist.destroy_process_group()
"""


def test_max_over_ranks_and_aggregate_two_gloo_ranks():
    import json
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER % ROOT], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    res = json.loads(outs[0][0].strip().splitlines()[-1])
    assert res["ms"] == 15.0 and res["e2e"] == 100.0              # the slowest rank sets the time
    assert res["value"] == 2 * 1000 * 4 / 15.0e-3                  # both replicas' cells count
    assert outs[1][0].strip() == ""                               # only rank 0 prints


def test_reference_arm_other_ranks_do_no_work():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"], env=env,
                       capture_output=True, text=True, timeout=240)
    assert p.returncode == 0 and p.stdout.strip() == ""
