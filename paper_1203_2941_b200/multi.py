"""Partitioned runs over several GPUs, one process per GPU (packets are independent).

Plumbing only -- every number is computed by the CUDA library:
  * each rank transports slice `rank` of `world` of EVERY epoch's packet ids (mcrt_run_begin / _step with
    part_index / part_count), on a replica of the grid and the tables;
  * after every epoch the ranks' integer tallies are summed (between epochs only the absorption counts, as the
    epoch's own increments; after the last epoch / every sweep also the Lucy tallies, the escape histograms and the
    run counters), so the next epoch's temperature update sees the global counts.  Integer sums are exact and
    order-independent: the result is bit-identical to the single-GPU run.

Two ways to do the sum:
  "p2p"   the library's own reduce-scatter / all-gather kernel (mcrt_exchange_peer_sum) reads and writes the
          peers' tallies directly over NVLink: every rank maps the other ranks' workspaces into its address space
          with CUDA IPC (all contexts have the same layout, so a peer's array sits at the same offset in its
          workspace).  Two host barriers per exchange keep the phases apart;
  "nccl"  ncclAllReduce(ncclSum) in place on views of the workspace tensor (torch.distributed).
"""
from __future__ import annotations

import ctypes as C

from . import binding as B


def _view_i64(ws, ptr, words):
    """int64 view of `words` 64-bit words at device address `ptr` inside the workspace tensor `ws`."""
    import torch

    off = int(ptr) - ws.data_ptr()
    assert 0 <= off and off + 8 * int(words) <= ws.numel() and off % 8 == 0
    return ws[off:off + 8 * int(words)].view(torch.int64)


class PeerMap:
    """The other ranks' workspaces mapped into this process (CUDA IPC over torch's storage sharing)."""

    def __init__(self, ctx, group=None):
        import torch
        import torch.distributed as dist

        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        ws = ctx.workspace
        handle = ws.untyped_storage()._share_cuda_()          # (device, handle, size, offset, ref handle, ...)
        mine = (handle, ws.storage_offset(), ws.numel())
        allh = [None] * self.world
        dist.all_gather_object(allh, mine, group=group)
        self.bases, self._keep = [], []
        for r, (h, off, n) in enumerate(allh):
            if r == self.rank:
                self.bases.append(ws.data_ptr())
                continue
            st = torch.UntypedStorage._new_shared_cuda(*h)     # cudaIpcOpenMemHandle, peer access enabled lazily
            t = torch.empty(0, dtype=torch.uint8, device=ws.device).set_(st, off, (n,))
            self._keep.append((st, t))
            self.bases.append(t.data_ptr())
        self.my_base = ws.data_ptr()

    def views(self, ex: B.Exchange):
        """The same exchange arrays on every rank: a peer's array sits at the same offset in its workspace."""
        out = []
        for base in self.bases:
            v = B.Exchange()
            v.n = ex.n
            for a in range(ex.n):
                v.ptr[a] = base + (int(ex.ptr[a]) - self.my_base)
                v.words[a] = ex.words[a]
            out.append(v)
        return out


def exchange(ctx, group=None, peers: PeerMap | None = None):
    """Sum the tallies of the step just run over all ranks (call on every rank)."""
    import torch
    import torch.distributed as dist

    ex = B.mcrt_exchange_begin(ctx.ctx)
    if peers is not None:
        views = peers.views(ex)
        for phase in (0, 1):
            torch.cuda.synchronize()          # my step / my phase 0 has finished ...
            dist.barrier(group=group)         # ... and so has everybody else's: peers' arrays may be read / are complete
            B.mcrt_exchange_peer_sum(ctx.ctx, peers.rank, views, phase)
        torch.cuda.synchronize()
        dist.barrier(group=group)             # nobody still reads my arrays when the next epoch adds to them
    else:
        for a in range(ex.n):
            dist.all_reduce(_view_i64(ctx.workspace, ex.ptr[a], ex.words[a]), op=dist.ReduceOp.SUM, group=group)
    B.mcrt_exchange_end(ctx.ctx)


def run_partitioned(ctx, n_packets, seed, group=None, peers: PeerMap | None = None, want_stats=True, on_step=None, **kw):
    """One run of n_packets packets shared by all ranks of `group`; returns the GLOBAL statistics (on every rank).
    on_step(done) is called after every step's exchange."""
    import torch.distributed as dist

    rank, world = dist.get_rank(group), dist.get_world_size(group)
    ctx.run_begin(n_packets, seed, part_index=rank, part_count=world, **kw)
    done = False
    while not done:
        done = ctx.run_step()
        exchange(ctx, group, peers)
        if on_step is not None:
            on_step(done)
    return ctx.run_end(want_stats)
