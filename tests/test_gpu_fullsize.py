"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

cfg 2 is checked in full against the oracle.  cfgs 3, 4, 5 (2e13 .. 1.4e15 flop) are checked on
a column sample with the full H: columns are independent (pin P7), so the oracle run on a
column subset -- each sampled column with its own full degree -- is an exact oracle for those
columns of the full GPU run.  The sample covers the first/last column, the first and last
column of the lowest and highest degree classes and columns either side of kernel tile edges.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_1805_10121_b200 as pkg
from paper_1805_10121_b200 import workloads as W
from cheb_closed_form import p_m, rel_fro

pytestmark = pytest.mark.gpu
TOL = {torch.complex128: 1e-12, torch.float64: 1e-12, torch.complex64: 1e-4, torch.float32: 1e-4}


def _host(x):
    return x.t().cpu().t().numpy()


def _run_full(w):
    V = W.empty_colmajor(w.N, w.ncols, w.dtype, w.H.device)
    V.copy_(w.V0)
    ws = torch.empty(pkg.chase_filter_workspace_bytes(w.N, w.ncols, w.dtype), dtype=torch.uint8, device=w.H.device)
    pkg.chase_filter_ws(w.H, V, w.degrees, w.a, w.b, w.lambda1, ws)
    torch.cuda.synchronize()
    return V


def _sample(w, extra=()):
    deg = w.degrees.numpy()
    n = w.ncols
    cols = {0, n - 1, 63, 64, 65, 127, 128, n // 2}
    for d in (deg.min(), deg.max()):
        idx = np.nonzero(deg == d)[0]
        cols.update((int(idx[0]), int(idx[-1])))
    cols.update(extra)
    return sorted(c for c in cols if 0 <= c < n)


def _check_sample(w, V, cols, max_oracle_degree=None):
    Hn = _host(w.H)
    deg = w.degrees.numpy()[cols]
    ref = oracle.chase_filter(Hn, _host(w.V0[:, cols]), deg, w.a, w.b, w.lambda1)
    got = _host(V[:, cols])
    tol = TOL[w.dtype]
    assert np.all(np.isfinite(got))
    assert rel_fro(got, ref) <= tol
    for j in range(len(cols)):
        assert np.linalg.norm(got[:, j] - ref[:, j]) <= 10 * tol * np.linalg.norm(ref[:, j]), cols[j]


def test_cfg2_full_size_full_oracle():
    w = W.make_config(2, device="cuda")
    V = _run_full(w)
    ref = oracle.chase_filter(_host(w.H), _host(w.V0), w.degrees.numpy(), w.a, w.b, w.lambda1)
    got = _host(V)
    assert rel_fro(got, ref) <= 1e-12
    err = np.linalg.norm(got - ref, axis=0) / np.linalg.norm(ref, axis=0)
    assert err.max() <= 1e-11


def test_cfg3_full_size_sampled():
    w = W.make_config(3, device="cuda")
    V = _run_full(w)
    _check_sample(w, V, _sample(w)[:8])


def test_cfg4_full_size_sampled():
    """The metric config.  Oracle on 6 sampled columns (degrees 8 .. 36) with the full 25.6 GB H."""
    w = W.make_config(4, device="cuda")
    V = _run_full(w)
    deg = w.degrees.numpy()
    lo = np.nonzero(deg == deg.min())[0]
    cols = sorted({0, int(lo[-1]), int(lo[-1]) + 1, 1000, w.ncols - 1})
    _check_sample(w, V, cols)


def test_cfg4_shape_diagonal_closed_form_full_size():
    """Property that holds at any size: H = diag(h) gives out[i,j] = p_{m_j}(h_i) V0[i,j] (pin P5),
    checked on EVERY element of a full cfg-4-shaped run (N=40000, 2000 columns, degrees 8..36)."""
    w = W.make_config(4, device="cuda", N=8, ncols=2000)         # degrees/bounds of cfg 4
    N = 40000
    g = torch.Generator(device="cuda").manual_seed(4242)
    h = torch.rand(N, dtype=torch.float64, device="cuda", generator=g) * 4.0 - 2.0
    H = W.empty_colmajor(N, N, torch.complex128, "cuda")
    H.zero_()
    H.diagonal().copy_(h.to(torch.complex128))
    V0 = W.gaussian_colmajor(N, 2000, torch.complex128, 4243, "cuda")
    big = W.Workload("diag", H, V0, w.degrees, w.a, w.b, w.lambda1, torch.complex128)
    V = _run_full(big)
    hn = h.cpu().numpy()
    got, v0 = _host(V), _host(V0)
    deg = w.degrees.numpy()
    for d in np.unique(deg):
        cols = np.nonzero(deg == d)[0]
        ref = p_m(int(d), hn, w.a, w.b, w.lambda1)[:, None] * v0[:, cols]
        assert rel_fro(got[:, cols], ref) <= 1e-12, d


def test_cfg5_full_size_sampled():
    w = W.make_config(5, device="cuda")
    V = _run_full(w)
    _check_sample(w, V, [0, 1500, w.ncols - 1])
