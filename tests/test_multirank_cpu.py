"""N > 1 path on CPU: two gloo ranks.  bench.py's whole-job reduction (time = max over ranks), and the partition
arithmetic of a run shared by several GPUs: with the library's own host
helpers every rank derives the same epoch schedule and the ranks' slices tile every epoch's packet ids."""
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
assert seeds == [4, 4]            # ONE run: every rank uses the same seed, packet ids tell the packets apart
# partition arithmetic (pure host functions of the CUDA library): every epoch's ids are tiled by the ranks' slices
from paper_1203_2941_b200 import binding as B
for n, b0, bmax, growth in ((100001, 0, 0, 0.0), (10**8, 0, 0, 0.0), (5000, 100, 700, 1.5), (7, 0, 0, 0.0)):
    sizes = B.mcrt_epoch_schedule(n, b0, bmax, growth)
    assert int(sizes.sum()) == n and (growth or all(int(sizes[i + 1]) in (int(sizes[i]) * 2, int(sizes[i]), n - int(sizes[:i + 1].sum())) for i in range(len(sizes) - 1)))
    mine = [B.mcrt_part_slice(int(be), rank, world) for be in sizes]
    both = [None] * world
    dist.all_gather_object(both, mine)
    first = 0
    for e, be in enumerate(sizes):
        lo0, hi0 = both[0][e]; lo1, hi1 = both[1][e]
        assert lo0 == 0 and hi0 == lo1 and hi1 == int(be), (e, both[0][e], both[1][e])   # the slices tile [0, B_e)
        assert abs((hi0 - lo0) - (hi1 - lo1)) <= 1                                       # and are balanced
        first += int(be)
    assert first == n
assert B.mcrt_epoch_schedule(10**8)[0] == 2**18 and int(B.mcrt_epoch_schedule(10**8).max()) == 2**22
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
