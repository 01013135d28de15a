"""CPU-only tests of the C-ABI library's host side: exported symbols, validation and error
codes (all rejected before any CUDA call), the scalar recurrence and the active-suffix
schedule (Alg. 4 l.2-5, 8, 11-14)."""
import ctypes
import os
import re

import numpy as np
import pytest
import torch

import oracle
import paper_1805_10121_b200 as pkg
from paper_1805_10121_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    declared = set()
    for name in sorted(os.listdir(os.path.join(ROOT, "include"))):       # product ABI + the bench/test hooks
        header = open(os.path.join(ROOT, "include", name)).read()
        header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
        declared |= set(re.findall(r"\b(chase_[a-z0-9_]+)\s*\(", header))
    assert declared == set(binding.EXPORTS)
    product = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "chase_filter.h")).read(), flags=re.S)
    for hook in ("chase_fp64_peak_probe", "chase_filter_launch_count", "chase_filter_step_plan"):
        assert hook not in product            # hooks live in chase_filter_bench.h, not in the product header
    lib = ctypes.CDLL(pkg.lib_path())
    for name in declared:
        assert hasattr(lib, name), name


def test_strerror_covers_codes():
    for code in range(0, -9, -1):
        assert pkg.chase_filter_strerror(code) != "unknown error"
    assert pkg.chase_filter_strerror(-99) == "unknown error"


def test_scalars_match_oracle_and_closed_form():
    a, b, l1, m = -1.7, 2.05, -2.0, 36
    alpha, beta, c = pkg.chase_filter_scalars(a, b, l1, m)
    _, oalpha, obeta, oc, _ = oracle.chase_scalars(a, b, l1, m)
    np.testing.assert_allclose(alpha[1:], oalpha[1:], rtol=1e-15)
    np.testing.assert_allclose(beta[1:], obeta[1:], rtol=1e-15)
    assert c == oc
    assert beta[1] == 0.0


@pytest.mark.parametrize("bounds", [(-1.0, -1.0, -2.0), (2.0, 1.0, -2.0), (-1.0, 2.0, -1.0),
                                    (-1.0, 2.0, 0.0), (float("nan"), 2.0, -2.0), (-1.0, float("inf"), -2.0)])
def test_scalars_reject_bad_bounds(bounds):
    a, b, l1 = bounds
    with pytest.raises(pkg.ChaseFilterError) as ei:
        pkg.chase_filter_scalars(a, b, l1, 4)
    assert ei.value.code == -2


def test_schedule():
    deg = [0, 0, 2, 2, 3, 6, 6]
    m_max, off = pkg.chase_filter_schedule(deg)
    assert m_max == 6
    expect = [sum(1 for d in deg if d < k) for k in range(1, 7)]
    assert list(off[1:]) == expect == [2, 2, 4, 5, 5, 5]
    assert pkg.chase_filter_schedule([])[0] == 0
    for bad in ([2, 1], [-1, 2], [4, 4, 2]):
        with pytest.raises(pkg.ChaseFilterError) as ei:
            pkg.chase_filter_schedule(bad)
        assert ei.value.code == -3


def _raw_ws(H=0x1000, N=64, V=0x2000, ncols=4, degrees=(2, 2, 4, 4), a=-1.0, b=2.0, l1=-2.0,
            dtype=3, ws=0x3000, ws_bytes=1 << 25):
    lib = pkg.load()
    deg = np.asarray(degrees, dtype=np.int32)
    return lib.chase_filter_ws(H, N, V, ncols, deg.ctypes.data if deg.size else None, a, b, l1, dtype,
                               ws, ws_bytes, None)


def test_validation_rejects_before_any_launch():
    # fake (never dereferenced) device pointers: every call below must return before touching CUDA
    assert _raw_ws(dtype=7) == -4
    assert _raw_ws(N=0) == -1
    assert _raw_ws(H=None) == -1
    assert _raw_ws(V=None) == -1
    assert _raw_ws(ncols=-1) == -1
    assert _raw_ws(a=2.5) == -2
    assert _raw_ws(l1=-0.5) == -2
    assert _raw_ws(degrees=(4, 2, 4, 4)) == -3
    assert _raw_ws(degrees=(-2, 2, 4, 4)) == -3
    assert _raw_ws(ws=None) == -5
    assert _raw_ws(ws_bytes=16) == -5
    assert _raw_ws(H=0x1008) == -6
    assert _raw_ws(ws=0x3004) == -6
    # nothing to do: success without a launch, even with no workspace
    before = pkg.chase_filter_launch_count()
    assert _raw_ws(degrees=(0, 0, 0, 0), ws=None, ws_bytes=0) == 0
    assert _raw_ws(ncols=0, degrees=(), V=None, ws=None, ws_bytes=0) == 0
    assert pkg.chase_filter_launch_count() == before


def test_workspace_bytes():
    import torch
    sk = 1024 + 160 * 128 * 1024                            # FP64 tensor path: stream-K flags + partial tiles
    assert pkg.chase_filter_workspace_bytes(40000, 2000, torch.complex128) == 40000 * 2000 * 16 + sk
    assert pkg.chase_filter_workspace_bytes(60000, 3000, torch.complex64) == 60000 * 3000 * 8 + 256
    assert pkg.chase_filter_workspace_bytes(3, 1, torch.float32) == 256
    assert pkg.load().chase_filter_workspace_bytes(10, 10, 9) == 0


def test_binding_rejects_cpu_tensors_no_fallback():
    import torch
    from paper_1805_10121_b200 import workloads as W
    w = W.make_config(2, N=32, ncols=4)
    with pytest.raises(ValueError):
        pkg.chase_filter(w.H, w.V0.clone(), w.degrees, w.a, w.b, w.lambda1)
    with pytest.raises(ValueError):     # row-major input is a layout error, not silently transposed
        pkg.chase_filter_host(torch.zeros(8, 8, dtype=torch.float64), torch.zeros(8, 2, dtype=torch.float64),
                              [2, 2], -1.0, 2.0, -2.0)


def test_product_does_not_import_oracle():
    pkgdir = os.path.join(ROOT, "paper_1805_10121_b200")
    for dirpath, _, files in os.walk(pkgdir):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "liboracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1805_10121_b200" not in src and "from paper_1805_10121_b200" not in src, f
            assert "#include \"chase" not in src, f


@pytest.mark.parametrize("dtype,bn,quarter,bk", [(torch.complex128, 64, 16, 16), (torch.float64, 128, 32, 32)])
def test_step_plan_covers_every_tile_slab_exactly_once(dtype, bn, quarter, bk):
    """chase_filter_step_plan (host model only, no CUDA): the column tiles cover [0, n) exactly; the
    data-parallel tiles plus the stream-K ranges cover every k-slab of every tile exactly once; ranges
    are contiguous and ascending (a CTA only ever waits on lower-numbered CTAs)."""
    for N in (64, 512, 4096, 40000):
        for n in list(range(1, 70)) + [96, 127, 128, 129, 255, 256, 257, 1400, 1867, 2000, 2999]:
            for sms in (148, 132):
                pl = pkg.chase_filter_step_plan(N, n, dtype, sms)
                w, tm, tn = pl["tile_width"], pl["tiles_m"], pl["tiles_n"]
                assert tm == -(-N // 128) and pl["slabs_per_tile"] == -(-N // bk)
                assert w % quarter == 0 and quarter <= w <= bn
                assert tn == -(-n // w), (N, n, w, tn)
                T, D, G, KT = tm * tn, pl["dp_tiles"], pl["sk_ctas"], pl["slabs_per_tile"]
                assert 0 <= D <= T and 0 <= G <= min(sms, 160)
                skb = pl["sk_begin"]
                grid, rounds = pl["grid"], pl["dp_rounds"]
                if G == 0:
                    assert D == T and grid == T and rounds == 1     # one CTA per tile
                    continue
                # whole tiles: CTA b owns r * grid + b < D for r < rounds -- every tile below D exactly once;
                # default plan: persistent CTAs (lock-step), stream-K ranges on the same CTAs
                first = pl["sk_first"]
                assert (rounds, first, grid) == ((D // sms, 0, sms) if D > 0 else (0, 0, G))
                assert D % sms == 0
                assert len(skb) == G + 1 and skb[0] == 0 and skb[-1] == (T - D) * KT
                assert np.all(np.diff(skb) >= 0)


def test_step_plan_balances_the_benchmark_configs():
    """Modelled makespan (quarter-slab units, one CTA per SM, dispatch in blockIdx order) of the plan
    vs the perfect split: cfg 1 (latency-bound: 16 tiles for 148 SMs), cfg 2 (128 tiles for 148 SMs),
    cfg 4 full width (10016 tiles, ragged last column tile)."""
    import heapq

    def makespan(N, n, dtype, sms=148):
        pl = pkg.chase_filter_step_plan(N, n, dtype, sms)
        cplx = dtype == torch.complex128
        warps_n, group_n = (2, 16) if cplx else (4, 12)
        w, tm, tn, KT = pl["tile_width"], pl["tiles_m"], pl["tiles_n"], pl["slabs_per_tile"]

        def quarters(t, ragged_last):                             # cost of one slab of raster tile t
            body_n = tn - 1 if ragged_last else tn                # lock-step plans: the ragged tile column comes last
            if t >= body_n * tm:
                col = body_n
            else:
                per_group = group_n * tm
                grp = t // per_group
                first = grp * group_n
                gn = min(group_n, body_n - first)
                col = first + (t - grp * per_group) % gn
            v = min(w, n - col * w)
            return -(-(-(-v // 8)) // warps_n)

        grid, rounds = pl["grid"], pl["dp_rounds"]
        busy = [0.0] * grid                                       # persistent CTAs, one per SM
        for r in range(rounds):
            for b in range(grid):
                t = r * grid + b
                if t < pl["dp_tiles"]:
                    busy[b] += quarters(t, rounds > 0) * KT
        skb = pl["sk_begin"]
        for g in range(pl["sk_ctas"]):
            s = int(skb[g])
            while s < skb[g + 1]:
                t = pl["dp_tiles"] + s // KT
                take = min(int(skb[g + 1]) - s, KT - s % KT)
                busy[g] += take * quarters(t, rounds > 0)
                s += take
        assert grid <= sms or pl["sk_ctas"] == 0
        return max(busy), sum(busy) / sms

    for N, n, dtype, slack in ((512, 60, torch.complex128, 1.10), (4096, 256, torch.complex128, 1.01),
                               (4096, 37, torch.complex128, 1.03), (40000, 2000, torch.complex128, 1.002),
                               (40000, 1867, torch.complex128, 1.002), (20000, 1400, torch.float64, 1.002)):
        end, ideal = makespan(N, n, dtype)
        assert end <= slack * ideal + 4, (N, n, end, ideal)


def test_rows_and_lanczos_validation_rejects_before_any_launch():
    """chase_hemm_rows / chase_filter_rows_ws / chase_rows_barrier / chase_lanczos: fake pointers, every call
    must come back with its error code before touching CUDA."""
    import ctypes as C
    lib = pkg.load()
    before = pkg.chase_filter_launch_count()
    H, X, Y = 0x1000, 0x2000, 0x3000
    peers = (C.c_void_p * 2)(0x4000, 0x5000)

    def hemm_rows(N=64, row0=0, nrows=32, ncols=4, dtype=3, npeers=0, peer=None, x=X, y=Y, alpha=1.0):
        return lib.chase_hemm_rows(H, N, row0, nrows, x, y, ncols, alpha, 0.0, 0.0, dtype, npeers, peer, None)

    assert hemm_rows(dtype=9) == -4
    assert hemm_rows(dtype=2) == -6                       # only the FP64 tensor kernels take row blocks
    assert hemm_rows(nrows=12) == -6                      # not a multiple of the 8-row group
    assert hemm_rows(row0=40, nrows=32) == -1             # block leaves the matrix
    assert hemm_rows(npeers=2, peer=None) == -1
    assert hemm_rows(npeers=16, peer=peers) == -1
    assert hemm_rows(y=X) == -1                           # in-place product is not defined
    assert hemm_rows(alpha=float("nan")) == -1
    assert hemm_rows(ncols=0) == 0
    assert hemm_rows(dtype=1, N=64, nrows=24) == -6       # f64: 16-row groups

    deg = np.asarray([2, 2, 4, 4], dtype=np.int32)
    seq = C.c_uint32(0)

    def rows_ws(nranks=1, rank=0, peer_v=None, peer_w=None, flags=None, peer_flags=None, a=-1.0, ws_bytes=1 << 20,
                degrees=deg):
        return lib.chase_filter_rows_ws(H, 64, 0, 32, X, 4, degrees.ctypes.data, a, 2.0, -2.0, 3, Y, ws_bytes,
                                        nranks, rank, peer_v, peer_w, flags, peer_flags, C.addressof(seq), None)

    assert rows_ws(nranks=0) == -1
    assert rows_ws(nranks=2, rank=2) == -1
    assert rows_ws(nranks=2, rank=0) == -1                # peers missing
    assert rows_ws(flags=0x6000, peer_flags=None) == -1
    assert rows_ws(a=3.0) == -2
    assert rows_ws(degrees=np.asarray([4, 2, 4, 4], dtype=np.int32)) == -3
    assert rows_ws(ws_bytes=16) == -5
    assert seq.value == 0                                 # no barrier was enqueued

    assert lib.chase_rows_barrier(None, peers, 2, 0, 1, None) == -1
    assert lib.chase_rows_barrier(0x6000, peers, 2, 5, 1, None) == -1
    assert lib.chase_rows_barrier(0x6000, peers, 17, 0, 1, None) == -1
    assert lib.chase_rows_signal(0x6000, None, 2, 0, 1, None) == -1
    assert lib.chase_rows_wait(None, 2, 1, None) == -1
    assert lib.chase_rows_wait(0x6000, 0, 1, None) == -1
    assert lib.chase_rows_status(None, 2, None) == -1
    assert lib.chase_rows_status(0x6000, 17, None) == -1
    cb = binding.HOST_BARRIER_FN(lambda _ctx: 0)
    assert lib.chase_filter_rows_hostsync_ws(H, 64, 0, 32, X, 4, deg.ctypes.data, -1.0, 2.0, -2.0, 3, Y, 1 << 20,
                                             1, 0, None, None, None, None, C.addressof(seq), None, cb, None) == -1   # host barrier without flags
    assert rows_ws(degrees=np.asarray([2, 2, 4, 5000], dtype=np.int32)) == -3     # above CHASE_MAX_DEGREE

    al = np.zeros(10)
    def lanczos(N=64, nruns=2, k=5, dtype=3, ws=0x7000, ws_bytes=1 << 24, v0=X):
        return lib.chase_lanczos(H, N, v0, nruns, k, dtype, al.ctypes.data, al.ctypes.data, ws, ws_bytes, None)
    assert lanczos(dtype=8) == -4
    assert lanczos(k=0) == -1
    assert lanczos(k=65) == -1                            # more steps than the dimension
    assert lanczos(nruns=0) == -1
    assert lanczos(v0=None) == -1
    assert lanczos(ws=None) == -5
    assert lanczos(ws_bytes=1024) == -5
    assert lanczos(ws=0x7008) == -6

    cnt = C.c_int64(-1)
    dst = np.asarray([0, 1], dtype=np.int64)
    def ritz_vecs(run=1, nruns=2, k=5, ws=0x7000, ws_bytes=1 << 24, vhat=Y, ncv=4, d=dst, mu=0.0):
        return lib.chase_lanczos_ritz_vectors(ws, ws_bytes, 64, nruns, k, 3, run, al.ctypes.data, al.ctypes.data, mu,
                                              vhat, ncv, d.ctypes.data, d.size, C.addressof(cnt), None, None)
    assert ritz_vecs(run=2) == -1                          # run out of range
    assert ritz_vecs(k=0) == -1
    assert ritz_vecs(vhat=None) == -1
    assert ritz_vecs(d=np.asarray([0, 4], dtype=np.int64)) == -1      # target column outside Vhat
    assert ritz_vecs(mu=float("nan")) == -1
    assert ritz_vecs(ws=None) == -5
    assert ritz_vecs(ws_bytes=64) == -5
    assert ritz_vecs(vhat=0x3008) == -6
    assert pkg.chase_filter_launch_count() == before


def test_parity_sample_plan_covers_every_degree_class_and_tile_edge():
    """>= 32 columns; first / last column of every distinct degree; global first / last;
    columns around the kernels' column-tile multiples; deterministic."""
    from paper_1805_10121_b200 import workloads as W
    for cfg in (3, 4, 5):
        shape = W.CONFIG_SHAPES[cfg]
        if cfg == 4:
            deg = W.sorted_even_degrees(shape["ncols"], 8, 36, W.BASE_SEED + 4002)
        else:
            deg = W.uniform_degrees(shape["ncols"], 20 if cfg == 3 else 16)
        cols = W.parity_sample_columns(deg)
        assert cols == W.parity_sample_columns(deg)
        assert cols == sorted(set(cols)) and len(cols) >= 32
        assert cols[0] == 0 and cols[-1] == shape["ncols"] - 1
        d = deg.numpy()
        for v in np.unique(d):
            idx = np.nonzero(d == v)[0]
            assert idx[0] in cols and idx[-1] in cols
        assert {63, 64, 65, 127, 128, 129} <= set(cols)
    assert W.parity_sample_columns([]) == []
    assert W.parity_sample_columns([2, 2, 4]) == [0, 1, 2]


def test_host_handle_rejects_bad_arguments_before_any_cuda_call():
    lib = pkg.load()
    out = ctypes.c_void_p()
    assert lib.chase_filter_host_open(None, 64, 8, binding.CHASE_C128, 0, ctypes.addressof(out)) == -1
    assert lib.chase_filter_host_open(0x1000, 64, 0, binding.CHASE_C128, 0, ctypes.addressof(out)) == -1
    assert lib.chase_filter_host_open(0x1000, 64, 8, 7, 0, ctypes.addressof(out)) == -4
    assert lib.chase_filter_host_run(None, 0x1000, 4, 0x2000, -1.0, 1.0, -2.0) == -1
    assert lib.chase_filter_host_close(None) == -1
