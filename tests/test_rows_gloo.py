"""Row-sharded multi-GPU path, host logic on CPU (world_size-2 gloo): the row partition and the peer
pointer table built from exchanged CUDA-IPC handles (the export / open calls are faked -- they need
GPUs -- the exchange protocol is the real one)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1805_10121_b200 import sharding


@pytest.mark.parametrize("N,world,align", [(40000, 8, 128), (40000, 3, 128), (520, 2, 8), (96, 4, 16), (128, 3, 128)])
def test_row_partition_covers_rows_once(N, world, align):
    parts = sharding.row_partition(N, world, align)
    assert len(parts) == world
    pos = 0
    for row0, nrows in parts:
        assert row0 == pos and nrows >= 0
        pos += nrows
        if row0 + nrows < N:
            assert nrows % align == 0
    assert pos == N
    sizes = [n for _, n in parts if n]
    assert max(sizes) - min(sizes) <= 2 * align or len(sizes) < world


class _FakeTensor:
    def __init__(self, ptr):
        self.ptr = ptr

    def data_ptr(self):
        return self.ptr


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # each "process" has V and W inside ONE allocation (base 0x1000 * (rank+1)) and flags in another
        base = 0x100000 * (rank + 1)
        tensors = {"V": _FakeTensor(base + 256), "W": _FakeTensor(base + 4096), "flags": _FakeTensor(base + 0x80000)}
        alloc_of = {"V": base, "W": base, "flags": base + 0x80000}

        def export(t):
            nm = next(k for k, v in tensors.items() if v is t)
            return (f"alloc-{alloc_of[nm]:x}".encode(), t.data_ptr() - alloc_of[nm])

        opened = []

        def open_handle(h):
            opened.append(h)
            return 0x7000000 + int(h.decode().split("-")[1], 16)     # the peer mapping lands elsewhere

        table, bases = sharding.exchange_peer_pointers(tensors, rank, world, export=export, open_handle=open_handle)
        np.save(os.path.join(out_dir, f"table{rank}.npy"),
                np.array([table["V"], table["W"], table["flags"]], dtype=np.int64))
        np.save(os.path.join(out_dir, f"opened{rank}.npy"), np.array([len(opened), len(bases)]))
    finally:
        dist.destroy_process_group()


def test_two_rank_peer_pointer_exchange(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    for rank in range(world):
        t = np.load(tmp_path / f"table{rank}.npy")
        peer = 1 - rank
        own_base, peer_base = 0x100000 * (rank + 1), 0x100000 * (peer + 1)
        assert list(t[:, rank]) == [own_base + 256, own_base + 4096, own_base + 0x80000]
        assert list(t[:, peer]) == [0x7000000 + peer_base + 256, 0x7000000 + peer_base + 4096,
                                    0x7000000 + peer_base + 0x80000 + 0]
        n_open, n_bases = np.load(tmp_path / f"opened{rank}.npy")
        assert n_open == 2 and n_bases == 2          # V and W share an allocation: mapped once
