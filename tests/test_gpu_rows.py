"""Row-sharded path on ONE GPU (SURVEY 8(e) option 2).  The P "ranks" are logical: each has its own row
block of H and its own full copies of the vector buffers on the same device, the peer pointers are
simply the other copies' addresses, and the ranks' launches are issued one after the other on one
stream (stream order stands in for the inter-GPU barrier; no kernel waits on another).  This checks
what the kernel does with row offsets, the rectangular H view and the peer stores; the flag barrier is
exercised with a single rank only."""
import numpy as np
import pytest
import torch

import oracle
import paper_1805_10121_b200 as pkg
from paper_1805_10121_b200 import sharding
from paper_1805_10121_b200 import workloads as W
from cheb_closed_form import rel_fro

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _dev(x):
    out = W.empty_colmajor(x.shape[0], x.shape[1], x.dtype, DEV)
    out.copy_(x)
    return out


def _row_blocks(H, world, align):
    parts = sharding.row_partition(H.shape[0], world, align)
    return parts, [_dev(H[r0:r0 + n, :]) for r0, n in parts]


@pytest.mark.parametrize("dtype,N,n,world,align", [(torch.complex128, 520, 77, 3, 128), (torch.float64, 1040, 150, 2, 128),
                                                    (torch.complex128, 776, 40, 4, 8), (torch.float64, 528, 33, 3, 16)])
def test_hemm_rows_with_peer_pushes(dtype, N, n, world, align):
    H = W.hermitian_gaussian_ensemble(N, dtype, seed=81)
    X = W.gaussian_colmajor(N, n, dtype, seed=82)
    Y = W.gaussian_colmajor(N, n, dtype, seed=83)
    parts, Hb = _row_blocks(H, world, align)
    Xs = [_dev(X) for _ in range(world)]
    Ys = [_dev(Y) for _ in range(world)]
    for r, (row0, nrows) in enumerate(parts):
        peers = [Ys[q].data_ptr() for q in range(world) if q != r]
        pkg.chase_hemm_rows(Hb[r], row0, Xs[r], Ys[r], alpha=0.7, beta=-1.3, shift=0.25, peer_Y=peers)
    torch.cuda.synchronize()
    ref = oracle.hemm(H.numpy(), X.numpy(), Y.numpy(), 0.7, -1.3, 0.25)
    for q in range(world):
        assert rel_fro(Ys[q].cpu().numpy(), ref) <= 1e-12, q


def test_hemm_rows_on_side_stream_with_cold_scratch_cache():
    """The row-sharded HEMM takes its stream-K scratch from the library's cache; a fresh buffer must be zeroed on
    the launching (non-blocking) stream, not on the legacy default stream."""
    dtype, N, n, world = torch.complex128, 520, 77, 3
    H = W.hermitian_gaussian_ensemble(N, dtype, seed=84)
    X = W.gaussian_colmajor(N, n, dtype, seed=85)
    parts, Hb = _row_blocks(H, world, 128)
    Xd = _dev(X)
    ref = oracle.hemm(H.numpy(), X.numpy(), None)
    torch.cuda.synchronize()
    for _ in range(3):
        pkg.chase_scratch_cache_release()
        st = torch.cuda.Stream()
        Yd = W.empty_colmajor(N, n, dtype, DEV)
        Yd.fill_(float("nan"))
        torch.cuda.synchronize()
        for r, (row0, nrows) in enumerate(parts):
            pkg.chase_hemm_rows(Hb[r], row0, Xd, Yd, stream=st)
        st.synchronize()
        assert rel_fro(Yd.cpu().numpy(), ref) <= 1e-12


@pytest.mark.parametrize("dtype,N,n,world", [(torch.complex128, 520, 77, 3), (torch.float64, 1040, 150, 2)])
def test_filter_emulated_ranks_step_by_step(dtype, N, n, world):
    """Alg. 4 driven from the host plan (chase_filter_scalars / _schedule) with one chase_hemm_rows per
    rank and step on the active suffix; every rank's copy of V must end up equal to the oracle."""
    w = W.make_config(2, N=N, ncols=n, dtype=dtype)
    deg = w.degrees.numpy()
    parts, Hb = _row_blocks(w.H, world, 128)
    buf = [[_dev(w.V0) for _ in range(world)], [_dev(torch.zeros_like(w.V0)) for _ in range(world)]]
    m_max, offset = pkg.chase_filter_schedule(deg)
    alpha, beta, c = pkg.chase_filter_scalars(w.a, w.b, w.lambda1, m_max)
    for k in range(1, m_max + 1):
        s, src = int(offset[k]), (k - 1) & 1
        for r, (row0, _) in enumerate(parts):
            X, Y = buf[src][r][:, s:], buf[src ^ 1][r][:, s:]
            peers = [buf[src ^ 1][q][:, s:].data_ptr() for q in range(world) if q != r]
            pkg.chase_hemm_rows(Hb[r], row0, X, Y, alpha=alpha[k], beta=beta[k] if k > 1 else 0.0, shift=c, peer_Y=peers)
    torch.cuda.synchronize()
    ref = oracle.chase_filter(w.H.numpy(), w.V0.numpy(), deg, w.a, w.b, w.lambda1)
    assert np.all(deg % 2 == 0)                      # even degrees: the result sits in buffer 0
    for q in range(world):
        assert rel_fro(buf[0][q].cpu().numpy(), ref) <= 1e-12, q


@pytest.mark.parametrize("with_flags", [False, True])
def test_filter_rows_single_rank_equals_plain_filter(with_flags):
    w = W.make_config(4, N=776, ncols=130)
    H = _dev(w.H)
    V1, V2 = _dev(w.V0), _dev(w.V0)
    ws = torch.empty(pkg.chase_filter_workspace_bytes(w.N, w.ncols, w.dtype), dtype=torch.uint8, device=DEV)
    pkg.chase_filter_ws(H, V1, w.degrees, w.a, w.b, w.lambda1, ws)
    flags = torch.zeros(2, dtype=torch.int32, device=DEV) if with_flags else None      # slot + status word
    seq = pkg.chase_filter_rows_ws(H, 0, V2, w.degrees, w.a, w.b, w.lambda1, ws, rank=0,
                                   flags=flags, peer_flags=[flags.data_ptr()] if with_flags else [], seq=5)
    torch.cuda.synchronize()
    assert torch.equal(V1, V2)
    if with_flags:
        m_max = int(w.degrees.max())
        assert seq == 5 + 1 + m_max and int(flags.cpu()[0]) == seq      # one barrier on entry, one per step
        pkg.chase_rows_status(flags, 1)                                 # no barrier timed out
        assert int(flags.cpu()[1]) == 0


def test_host_barrier_exception_is_not_swallowed():
    """A host barrier that raises (peer died, gloo timeout) must surface as that exception, at once -- not as a
    success that sends the run into the wait kernel's 30 s timeout."""
    import time
    w = W.make_config(4, N=520, ncols=24)
    H, V = _dev(w.H), _dev(w.V0)
    ws = torch.empty(pkg.chase_filter_workspace_bytes(w.N, w.ncols, w.dtype), dtype=torch.uint8, device=DEV)
    flags = torch.zeros(2, dtype=torch.int32, device=DEV)
    calls = []

    def barrier():
        calls.append(1)
        if len(calls) == 2:
            raise RuntimeError("peer died")
        return 0

    t0 = time.perf_counter()
    with pytest.raises(RuntimeError, match="peer died"):
        pkg.chase_filter_rows_ws(H, 0, V, w.degrees, w.a, w.b, w.lambda1, ws, rank=0, flags=flags,
                                 peer_flags=[flags.data_ptr()], seq=0, host_barrier=barrier)
    torch.cuda.synchronize()
    assert len(calls) == 2 and time.perf_counter() - t0 < 5.0
    # a barrier that merely REPORTS failure still maps to CHASE_ERR_TIMEOUT
    flags.zero_()
    with pytest.raises(pkg.ChaseFilterError) as e:
        pkg.chase_filter_rows_ws(H, 0, V, w.degrees, w.a, w.b, w.lambda1, ws, rank=0, flags=flags,
                                 peer_flags=[flags.data_ptr()], seq=0, host_barrier=lambda: 3)
    assert e.value.code == -7
    torch.cuda.synchronize()


def test_rows_rejects_unsupported_layouts():
    H = _dev(W.hermitian_gaussian_ensemble(64, torch.complex64, seed=1))
    X = _dev(W.gaussian_colmajor(64, 4, torch.complex64, seed=2))
    with pytest.raises(pkg.ChaseFilterError) as e:
        pkg.chase_hemm_rows(H, 0, X, X.clone())
    assert e.value.code == -6
    H = _dev(W.hermitian_gaussian_ensemble(520, torch.complex128, seed=1))
    X = _dev(W.gaussian_colmajor(520, 4, torch.complex128, seed=2))
    with pytest.raises(pkg.ChaseFilterError) as e:       # 100 rows: not a multiple of 8
        pkg.chase_hemm_rows(W.as_colmajor(H[:100, :]), 0, X, X.clone())
    assert e.value.code == -6


def test_row_sharded_filter_class_single_rank():
    """RowShardedFilter with world = 1 (no IPC): same result as the oracle, barrier sequence advances."""
    w = W.make_config(2, N=520, ncols=40)
    f = sharding.RowShardedFilter(_dev(w.H), 0, w.N, w.ncols, rank=0, world=1)
    f.V.copy_(w.V0)
    f.run(w.degrees, w.a, w.b, w.lambda1)
    torch.cuda.synchronize()
    ref = oracle.chase_filter(w.H.numpy(), w.V0.numpy(), w.degrees.numpy(), w.a, w.b, w.lambda1)
    assert rel_fro(f.V.cpu().numpy(), ref) <= 1e-12
    assert f.seq == 1 + int(w.degrees.max())
    f.close()


def test_barrier_whose_peer_never_signals_fails_loudly(monkeypatch):
    """A dead peer must not produce CHASE_OK: the wait kernel gives up after the (overridden, short)
    timeout, sets the sticky status word, later waits return at once, and chase_rows_status raises
    CHASE_ERR_TIMEOUT (-7).  One kernel polls alone for 100 ms; nothing waits on another kernel."""
    monkeypatch.setenv("CHASE_ROWS_TIMEOUT_MS", "100")
    flags = torch.zeros(3, dtype=torch.int32, device=DEV)            # 2 ranks + status word
    dead_peer = torch.zeros(3, dtype=torch.int32, device=DEV)        # rank 1's array; rank 1 never runs
    peers = [flags.data_ptr(), dead_peer.data_ptr()]
    import time
    t0 = time.perf_counter()
    pkg.chase_rows_barrier(flags, peers, rank=0, seq=1)
    pkg.chase_rows_barrier(flags, peers, rank=0, seq=2)              # returns at once: status already set
    with pytest.raises(pkg.ChaseFilterError) as e:
        pkg.chase_rows_status(flags, 2)
    dt = time.perf_counter() - t0
    assert e.value.code == -7
    assert 0.05 < dt < 5.0, dt
    f = flags.cpu().numpy()
    assert f[0] == 2 and f[1] == 0 and f[2] == 1                     # own slot signalled, peer silent, failed at seq 1
    assert int(dead_peer.cpu()[0]) == 2                              # the signal did reach the peer's array
    # a filter on these flags reports the failure too
    w = W.make_config(2, N=520, ncols=16)
    H, V = _dev(w.H), _dev(w.V0)
    ws = torch.empty(pkg.chase_filter_workspace_bytes(w.N, w.ncols, w.dtype), dtype=torch.uint8, device=DEV)
    other_V, other_W = _dev(w.V0), _dev(w.V0)
    pkg.chase_filter_rows_ws(H, 0, V, w.degrees, w.a, w.b, w.lambda1, ws, rank=0,
                             peer_V=[0, other_V.data_ptr()], peer_W=[0, other_W.data_ptr()],
                             flags=flags, peer_flags=peers, seq=2)
    with pytest.raises(pkg.ChaseFilterError) as e:
        pkg.chase_rows_status(flags, 2)
    assert e.value.code == -7


def _two_process_worker(rank, world, port, N, n, dtype_name, q):
    """One REAL process per rank, both on cuda:0: real chase_ipc_export / chase_ipc_open of the peer's V,
    W and flag arrays, real peer stores from the step kernel's epilogue, real flag signals and waits.
    The ranks time-share the GPU, so the barrier is host-sequenced (chase_filter_rows_hostsync_ws:
    signal, stream sync, gloo barrier, wait) -- no kernel ever spins on a kernel of the other process."""
    import os
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        torch.cuda.set_device(0)
        dtype = getattr(torch, dtype_name)
        w = W.make_config(2, N=N, ncols=n, dtype=dtype)
        parts = sharding.row_partition(N, world, 128)
        row0, nrows = parts[rank]
        H_loc = _dev(w.H[row0:row0 + nrows, :])
        f = sharding.RowShardedFilter(H_loc, row0, N, n, rank, world, host_barrier=dist.barrier)
        f.V.copy_(w.V0)
        f.W.fill_(float("nan"))
        torch.cuda.synchronize()
        dist.barrier()
        f.run(w.degrees, w.a, w.b, w.lambda1)
        torch.cuda.synchronize()
        ref = oracle.chase_filter(w.H.numpy(), w.V0.numpy(), w.degrees.numpy(), w.a, w.b, w.lambda1)
        err = rel_fro(f.V.cpu().numpy(), ref)
        flags = f.flags.cpu().numpy().tolist()
        dist.barrier()
        f.close()
        q.put((rank, float(err), f.seq, flags))
    except Exception as exc:       # surface the failure in the parent instead of a hang
        q.put((rank, repr(exc), -1, []))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("dtype_name,N,n", [("complex128", 520, 77), ("float64", 1040, 150)])
def test_row_sharded_filter_two_real_processes_on_one_gpu(dtype_name, N, n):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29650 + (N % 97)
    procs = [ctx.Process(target=_two_process_worker, args=(r, 2, port, N, n, dtype_name, q)) for r in range(2)]
    for p in procs:
        p.start()
    results = []
    try:
        for _ in procs:
            results.append(q.get(timeout=300))
    finally:
        for p in procs:
            p.join(timeout=60)
            if p.is_alive():
                p.kill()
    w = W.make_config(2, N=N, ncols=n, dtype=getattr(torch, dtype_name))
    m_max = int(w.degrees.max())
    assert sorted(r[0] for r in results) == [0, 1]
    for rank, err, seq, flags in results:
        assert isinstance(err, float), err
        assert err <= 1e-12, (rank, err)
        assert seq == 1 + m_max
        assert flags[:2] == [seq, seq] and flags[2] == 0, flags      # both ranks' signals arrived; no timeout
