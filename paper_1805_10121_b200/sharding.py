"""Column sharding for multi-GPU runs.

Columns of the filter are independent (each output column depends only on H, its own input
column and its own degree), so N GPUs shard the COLUMNS and replicate H: no data-path
collective.  Columns arrive sorted by ascending degree (Alg. 1 l.15); dealing
them round-robin keeps every shard sorted and balances sum(deg) -- and therefore flops
(8 N^2 sum(deg)) -- to within one column per distinct degree.
"""
from __future__ import annotations

import numpy as np


def shard_columns(ncols: int, world: int, rank: int) -> np.ndarray:
    """Indices (ascending) of the columns owned by `rank`: rank, rank + world, ..."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("need 0 <= rank < world")
    return np.arange(rank, ncols, world, dtype=np.int64)


def unshard_columns(ncols: int, world: int) -> np.ndarray:
    """perm such that concat(shard_0, ..., shard_{world-1})[:, perm] is in the original order."""
    order = np.concatenate([shard_columns(ncols, world, r) for r in range(world)])
    perm = np.empty(ncols, dtype=np.int64)
    perm[order] = np.arange(ncols)
    return perm


def shard_balance(degrees, world: int):
    """sum(deg) per rank -- what each GPU's flop count is proportional to."""
    deg = np.asarray(degrees)
    return [int(deg[shard_columns(len(deg), world, r)].sum()) for r in range(world)]


# ---------------------------------------------------------------------------------------------
# Row sharding (option 2): for an H that exceeds one GPU.  Rank r owns the
# row block [row0, row0 + nrows) of H and a full copy of the vectors; chase_filter_rows_ws pushes
# each new row block into the peers' copies from the step kernel's epilogue.
# ---------------------------------------------------------------------------------------------
def row_partition(N: int, world: int, align: int = 128):
    """[(row0, nrows)] per rank: contiguous blocks, every block a multiple of `align` rows except that
    the last one takes the remainder (N itself must be a multiple of the kernel's row group)."""
    if world < 1 or N < 1 or align < 1:
        raise ValueError("need world >= 1, N >= 1, align >= 1")
    groups = -(-N // align)
    base, extra = divmod(groups, world)
    parts, row0 = [], 0
    for r in range(world):
        g = base + (1 if r < extra else 0)
        nrows = min(g * align, N - row0)
        parts.append((row0, max(nrows, 0)))
        row0 += max(nrows, 0)
    return parts


def exchange_peer_pointers(tensors, rank: int, world: int, export=None, open_handle=None, all_gather=None):
    """Builds, for every named device tensor, the table of device pointers to ALL ranks' instances of it
    (own entry: the tensor's own pointer; others: CUDA-IPC mappings).  Returns (table, bases) with
    table[name][q] an int pointer and `bases` the mapped allocation bases to close at teardown.
    `export`, `open_handle`, `all_gather` are injectable for CPU tests."""
    if export is None or open_handle is None:
        from . import binding
        export = export or binding.chase_ipc_export
        open_handle = open_handle or binding.chase_ipc_open
    if all_gather is None:
        import torch.distributed as dist

        def all_gather(obj):
            out = [None] * world
            dist.all_gather_object(out, obj)
            return out
    names = sorted(tensors)
    mine = {nm: export(tensors[nm]) for nm in names}                  # (handle, offset) per tensor
    everyone = all_gather(mine)
    table, bases, opened = {nm: [0] * world for nm in names}, [], {}
    for q in range(world):
        for nm in names:
            if q == rank:
                table[nm][q] = int(tensors[nm].data_ptr())
                continue
            handle, offset = everyone[q][nm]
            key = (q, handle)
            if key not in opened:                                      # one mapping per peer allocation
                opened[key] = int(open_handle(handle))
                bases.append(opened[key])
            table[nm][q] = opened[key] + int(offset)
    return table, bases


class RowShardedFilter:
    """One rank of a row-sharded filter (one process per GPU, torch.distributed initialised, NVLink peer
    access between the GPUs).  Owns the rank's row block of H, full V / scratch buffers and the barrier
    flags, exchanges CUDA-IPC handles once, then `run()` is one chase_filter_rows_ws call per filter.

        f = RowShardedFilter(H_loc, row0, N, ncols, rank, world)
        f.V.copy_(V0)                    # every rank fills the complete V0
        f.run(degrees, a, b, lambda1)    # f.V then holds the complete result on every rank

    `host_barrier` (a callable, e.g. torch.distributed.barrier over gloo) must be given when several
    ranks share ONE GPU: their kernels time-slice, so the inter-GPU barrier is then sequenced on the host
    (chase_filter_rows_hostsync_ws) instead of by a spinning kernel.  run() ends with chase_rows_status:
    a barrier that timed out raises instead of returning a half-gathered result.
    """

    def __init__(self, H_loc, row0: int, N: int, ncols: int, rank: int, world: int, host_barrier=None):
        import torch
        from . import binding, workloads
        self.binding = binding
        self.H_loc, self.row0, self.N, self.ncols, self.rank, self.world = H_loc, row0, N, ncols, rank, world
        dev, dtype = H_loc.device, H_loc.dtype
        self.V = workloads.empty_colmajor(N, ncols, dtype, dev)
        self.W = workloads.empty_colmajor(N, ncols, dtype, dev)
        self.flags = torch.zeros(world + 1, dtype=torch.int32, device=dev)    # arrival slots + sticky status word
        self.seq = 0
        self.host_barrier = host_barrier
        if world > 1:
            with torch.cuda.device(dev):
                self.table, self._bases = exchange_peer_pointers(
                    {"V": self.V, "W": self.W, "flags": self.flags}, rank, world)
        else:
            self.table = {"V": [self.V.data_ptr()], "W": [self.W.data_ptr()], "flags": [self.flags.data_ptr()]}
            self._bases = []

    def run(self, degrees, a: float, b: float, lambda1: float, stream=None):
        ws = self.W.t().view(-1).view(self._byte_dtype())     # W.t() is the contiguous (ncols, N) storage
        self.seq = self.binding.chase_filter_rows_ws(
            self.H_loc, self.row0, self.V, degrees, a, b, lambda1, ws, rank=self.rank,
            peer_V=self.table["V"], peer_W=self.table["W"], flags=self.flags,
            peer_flags=self.table["flags"], seq=self.seq, stream=stream, host_barrier=self.host_barrier)
        self.binding.chase_rows_status(self.flags, self.world, stream)        # raises on a timed-out barrier
        return self.V

    @staticmethod
    def _byte_dtype():
        import torch
        return torch.uint8

    def close(self):
        for b in self._bases:
            self.binding.chase_ipc_close(b)
        self._bases = []
