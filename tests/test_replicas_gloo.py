"""bench.py --gpus N runs N independent replicas: the only cross-rank step is the
max-over-ranks of the timed region.  Exercised here with two gloo processes on the CPU."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, sys.argv[1])
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = bench.max_over_ranks(1.0 + rank, dist, "cpu")          # rank 1 is the slow one
assert ms == 2.0, ms
assert bench.max_over_ranks(3.5, None, "cpu") == 3.5          # single process: unchanged
if rank == 0:
    print("VALUE", bench.replica_throughput(world, ms))
dist.barrier()
dist.destroy_process_group()
"""


def test_two_replicas_report_the_slowest_rank_and_the_aggregate_rate(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script), ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=180) for p in procs]
    for p, (out, err) in zip(procs, outs):
        assert p.returncode == 0, err
    assert "VALUE 1000.0" in outs[0][0]                       # 2 replicas / 2 ms per step
