"""Seeded random shapes through every kernel family against the oracle: N, ncols, dtype, degree mix
(including 0, odd, long runs of equal degrees) drawn at random, so that tile edges, narrow tiles, the
2-D / 3-D H views, the persistent tf32 rounds and the generic fall-backs all get hit at sizes nobody
hand-picked.  Small sizes: the oracle stays cheap."""
import numpy as np
import pytest
import torch

import oracle
import paper_1805_10121_b200 as pkg
from paper_1805_10121_b200 import workloads as W
from cheb_closed_form import rel_fro

pytestmark = pytest.mark.gpu
DTYPES = [torch.complex128, torch.float64, torch.complex64, torch.float32]
TOL = {torch.complex128: 1e-12, torch.float64: 1e-12, torch.complex64: 1e-4, torch.float32: 1e-4}


def _case(i):
    rng = np.random.default_rng(1805_10121 + i)
    dtype = DTYPES[i % 4]
    N = int(rng.integers(16, 900))
    if rng.random() < 0.5:
        N = (N // 16) * 16 + int(rng.choice([0, 2, 4, 8]))          # mostly sizes the tensor paths take
    N = max(N, 16)
    ncols = int(rng.choice([1, 2, 7, 8, 9, 15, 16, 17, 31, 33, 63, 64, 65, 100, 129, 200, 257]))
    kinds = rng.integers(0, 3)
    if kinds == 0:
        deg = np.sort(rng.integers(0, 11, size=ncols))
    elif kinds == 1:
        deg = np.full(ncols, int(rng.integers(1, 9)))
    else:
        deg = np.sort(rng.choice([2, 4, 6, 8], size=ncols))
    return dtype, N, ncols, deg.astype(np.int32)


@pytest.mark.parametrize("i", range(64))
def test_random_shape_against_oracle(i):
    dtype, N, ncols, deg = _case(i)
    w = W.make_config(2, N=N, ncols=ncols, dtype=dtype)
    H = W.empty_colmajor(N, N, dtype, "cuda"); H.copy_(w.H)
    V = W.empty_colmajor(N, ncols, dtype, "cuda"); V.copy_(w.V0)
    ws = torch.empty(max(pkg.chase_filter_workspace_bytes(N, ncols, dtype), 16), dtype=torch.uint8, device="cuda")
    ws.fill_(0xFF)
    pkg.chase_filter_ws(H, V, deg, w.a, w.b, w.lambda1, ws)
    torch.cuda.synchronize()
    got = V.cpu().numpy()
    ref = oracle.chase_filter(w.H.numpy(), w.V0.numpy(), deg, w.a, w.b, w.lambda1)
    assert np.all(np.isfinite(got)), (dtype, N, ncols)
    tol = TOL[dtype]
    nr = np.linalg.norm(ref, axis=0)
    err = np.linalg.norm(got - ref, axis=0)
    assert rel_fro(got, ref) <= tol, (dtype, N, ncols, pkg.chase_filter_kernel_path(N, ncols, dtype))
    assert np.all(err <= 10 * tol * np.maximum(nr, 1e-300)), (dtype, N, ncols, int(np.argmax(err / np.maximum(nr, 1e-300))))
    assert np.array_equal(got[:, deg == 0], w.V0.numpy()[:, deg == 0])
    assert torch.equal(H.cpu(), w.H)
