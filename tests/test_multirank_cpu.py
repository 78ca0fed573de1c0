"""N > 1 path of bench.py on CPU: two gloo ranks, the whole-job reduction (time = max over ranks, units summed)
and the per-rank replica seeds (independent replicas, no data-path collective)."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
import torch, torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
ms, counts = bench.reduce_over_ranks(10.0 + 5.0 * rank, [100 * (rank + 1), 7, rank], torch.device("cpu"), world)
assert ms == 15.0, ms
assert counts == [300.0, 14.0, 1.0], counts
seeds = [None] * world
dist.all_gather_object(seeds, bench.replica_seed(4, rank))
assert seeds == [4, 1004] and len(set(seeds)) == world
# the reference arm prints on rank 0 only
dist.barrier()
dist.destroy_process_group()
print("rank", rank, "ok")
'''


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_rank_reduction_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script), ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=240)[0] for p in procs]
    for rank, (p, out) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, out
        assert f"rank {rank} ok" in out


def test_single_rank_reduction_is_identity():
    sys.path.insert(0, ROOT)
    import torch

    import bench

    ms, counts = bench.reduce_over_ranks(3.5, [1, 2, 3], torch.device("cpu"), 1)
    assert ms == 3.5 and counts == [1.0, 2.0, 3.0]
