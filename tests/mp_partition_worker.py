"""Worker of tests/test_gpu_parity.py::test_partitioned_run_across_processes -- launched by torch.distributed.run
with 2 ranks that share ONE GPU (gloo for the host-side plumbing).  Each rank owns a context; the tallies are
summed after every epoch either by the library's peer-memory kernel over CUDA-IPC mapped workspaces ("p2p") or by
all_reduce on views of the workspace ("allreduce": the code path bench.py uses with NCCL on several GPUs).  The
result must be bit-identical to an unpartitioned run.  No kernel ever waits for another rank: the ranks meet at
host barriers only."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    import torch
    import torch.distributed as dist

    from paper_1203_2941_b200 import binding as B, multi, workloads as W

    mode = sys.argv[1]
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    torch.cuda.set_device(0)
    w = W.torus256(n_clumps=300, n=48)
    N, seed = 80_001, 91
    c = B.Context(w, device="cuda:0")
    peers = multi.PeerMap(c) if mode == "p2p" else None
    st = multi.run_partitioned(c, N, seed, peers=peers)
    raw = c.read_raw()
    st2 = multi.run_partitioned(c, N, seed, peers=peers, mode=B.MCRT_MODE_FROZEN_T_SWEEP, n_sweeps=2)
    raw2 = c.read_raw()
    ok = True
    if rank == 0:
        ref = B.Context(w, device="cuda:0")
        rs = ref.run(N, seed)
        rr = ref.read_raw()
        rs2 = ref.run(N, seed, mode=B.MCRT_MODE_FROZEN_T_SWEEP, n_sweeps=2)
        rr2 = ref.read_raw()
        for a, b, s, t in ((raw, rr, st, rs), (raw2, rr2, st2, rs2)):
            for key in ("k", "lucy_fx", "sed", "sed_direct", "tidx"):
                ok &= bool(np.array_equal(a[key], b[key]))
            for key in ("packets", "crossings", "dusty_crossings", "scatterings", "absorptions", "direct_escapes"):
                ok &= s[key] == t[key]
        ref.close()
    # every rank holds the same (global) tallies
    mine = torch.from_numpy(raw2["lucy_fx"].copy())
    both = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(both, mine)
    ok &= bool(torch.equal(both[0], both[1]))
    flag = torch.tensor([1 if ok else 0])
    dist.all_reduce(flag, op=dist.ReduceOp.MIN)
    dist.barrier()
    peers = None
    c.close()
    dist.destroy_process_group()
    if rank == 0:
        print("PARTITION_OK" if int(flag) == 1 else "PARTITION_MISMATCH", mode, flush=True)
    sys.exit(0 if int(flag) == 1 else 1)


if __name__ == "__main__":
    main()
