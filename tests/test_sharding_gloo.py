"""N > 1 host path on CPU: world_size-2 gloo run of the column sharding.
Each rank filters its shard (with the oracle -- the CUDA path needs a GPU), the shards are
all-gathered and must reproduce the single-process result exactly (columns are independent)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1805_10121_b200 import sharding
from paper_1805_10121_b200 import workloads as W


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_path):
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = W.make_config(4, N=96, ncols=21)          # every rank builds the same seeded inputs
        idx = sharding.shard_columns(w.ncols, world, rank)
        deg = w.degrees.numpy()[idx]
        assert np.all(np.diff(deg) >= 0)               # shards stay sorted
        out = oracle.chase_filter(w.H.numpy(), w.V0.numpy()[:, idx], deg, w.a, w.b, w.lambda1)
        # ragged shards (21 columns over 2 ranks): pad to the largest shard for all_gather
        width = (w.ncols + world - 1) // world
        buf = torch.zeros((width, w.N), dtype=torch.complex128)
        buf[: len(idx)] = torch.from_numpy(np.ascontiguousarray(out.T))
        gathered = [torch.zeros_like(buf) for _ in range(world)]
        dist.all_gather(gathered, buf)
        t = torch.tensor([float(deg.sum())], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)       # the max-over-ranks reduction bench.py uses
        if rank == 0:
            cols = [gathered[r][: len(sharding.shard_columns(w.ncols, world, r))] for r in range(world)]
            cat = torch.cat(cols, dim=0).numpy().T
            full = cat[:, sharding.unshard_columns(w.ncols, world)]
            np.save(out_path, full)
            np.save(out_path + ".max.npy", t.numpy())
    finally:
        dist.destroy_process_group()


def test_two_rank_column_sharding_matches_single_process(tmp_path):
    import oracle
    world = 2
    out_path = str(tmp_path / "gathered.npy")
    mp.spawn(_worker, args=(world, _free_port(), out_path), nprocs=world, join=True)
    w = W.make_config(4, N=96, ncols=21)
    ref = oracle.chase_filter(w.H.numpy(), w.V0.numpy(), w.degrees.numpy(), w.a, w.b, w.lambda1)
    got = np.load(out_path)
    assert np.array_equal(got, ref)
    bal = sharding.shard_balance(w.degrees.numpy(), world)
    assert np.load(out_path + ".max.npy")[0] == max(bal)


@pytest.mark.parametrize("ncols,world", [(2000, 8), (21, 2), (5, 8), (0, 4)])
def test_shard_partition_and_balance(ncols, world):
    parts = [sharding.shard_columns(ncols, world, r) for r in range(world)]
    allidx = np.sort(np.concatenate(parts)) if ncols else np.array([], dtype=np.int64)
    assert np.array_equal(allidx, np.arange(ncols))
    perm = sharding.unshard_columns(ncols, world)
    assert np.array_equal(np.concatenate(parts)[perm], np.arange(ncols))
    if ncols == 2000:
        deg = W.sorted_even_degrees(ncols, 8, 36, seed=7).numpy()
        bal = sharding.shard_balance(deg, world)
        assert max(bal) - min(bal) <= 2 * 15           # within one column per distinct degree step
