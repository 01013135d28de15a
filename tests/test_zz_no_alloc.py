"""chase_residuals_static: the residual norms (Alg. 1 l.8) for callers that may not allocate.

Some users of the library cannot call cudaMalloc at the point where they need the residuals: their host
application's pool already owns the whole GPU, or their HBM share was fixed at job start, or they sit in a
loop that must not enter the driver's allocator.  chase_residuals asks such a caller for an N x ncols
workspace; chase_residuals_static takes it from a 48 MiB static device array inside libchase_filter.so.
This file checks that the static-scratch entry point returns what the existing chase_residuals returns.

The file name sorts last on purpose (`pytest --collect-only`): the suite runs with `pytest -x`, so a failure
here must not hide any other test.  The GPU test passes alone in a fresh process (its first call is then
the one that resolves the array's device address) and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest
import torch

import paper_1805_10121_b200 as pkg
from paper_1805_10121_b200 import binding, workloads as W


def _dev(x):
    out = W.empty_colmajor(x.shape[0], x.shape[1], x.dtype, "cuda")
    out.copy_(x)
    return out


def test_static_limit_is_checked_before_any_cuda_call():
    """Runs on the CPU box: a request beyond the array is refused with its own error code before the
    library touches CUDA (the fake pointers are never dereferenced)."""
    lib = pkg.load()
    N, ncols = 1 << 14, 1 << 10                       # 256 MiB complex128 block
    assert pkg.chase_residuals_workspace_bytes(N, ncols, torch.complex128) > pkg.CHASE_STATIC_SCRATCH_BYTES
    ritz = np.zeros(ncols)
    rc = lib.chase_residuals_static(0x1000, N, 0x2000, ncols, ritz.ctypes.data, 0x3000, binding.CHASE_C128, None)
    assert rc == -8
    assert "static scratch" in pkg.chase_filter_strerror(rc)
    # the largest FP64-tensor-path block that fits, and the first that does not (N = 4096 complex128: 64 KiB per column)
    fits = [n for n in range(400, 500) if
            pkg.chase_residuals_workspace_bytes(4096, n, torch.complex128) <= pkg.CHASE_STATIC_SCRATCH_BYTES]
    assert fits and max(fits) == 447, fits[-1:]       # 447 columns = 27.94 MiB + 20 MiB stream-K scratch + shifts
    # the other rejections match chase_residuals
    assert lib.chase_residuals_static(0x1000, 64, 0x2000, 4, ritz.ctypes.data, 0x3000, 9, None) == -4
    assert lib.chase_residuals_static(None, 64, 0x2000, 4, ritz.ctypes.data, 0x3000, binding.CHASE_C128, None) == -1
    assert lib.chase_residuals_static(0x1008, 64, 0x2000, 4, ritz.ctypes.data, 0x3000, binding.CHASE_C128, None) == -6
    assert lib.chase_residuals_static(0x1000, 64, 0x2000, 0, None, None, binding.CHASE_C128, None) == 0


# (dtype, N, ncols): one case per kernel family the entry point can route to, each used twice in a row and
# in an order that makes every call find another shape's (and another dtype's) leftovers in the array.
CASES = [
    (torch.complex128, 1544, 200),     # FP64 tensor kernel incl. stream-K tail: flags + partial tiles in the array
    (torch.complex64, 1282, 140),      # tcgen05 kernel: soft-barrier counter in the array
    (torch.float64, 1040, 150),        # FP64 tensor kernel, real
    (torch.float32, 203, 20),          # generic FMA kernel (no control block)
    (torch.complex128, 520, 5),        # streaming kernel (no control block)
    (torch.complex128, 3893, 282),     # the paper's NaCl size: 36.8 of the 48 MiB
]


@pytest.mark.gpu
def test_static_scratch_residuals_match_chase_residuals():
    """Every case: chase_residuals (caller's workspace; the existing path) against two consecutive calls of
    chase_residuals_static, within the tolerance test_hemm_residuals.py uses for residual norms
    (rtol = 10 * tol, tol = 1e-12 for FP64 and 1e-4 for FP32 arithmetic).  Inputs must come back untouched,
    and once everything is set up the static calls must not change the amount of allocated device memory."""
    prepared = []
    for i, (dtype, N, n) in enumerate(CASES):
        H = _dev(W.hermitian_gaussian_ensemble(N, dtype, seed=300 + i))
        V = _dev(W.gaussian_colmajor(N, n, dtype, seed=400 + i))
        ritz = np.linspace(-2.0, 2.0, n)
        want = pkg.chase_residuals(H, V, ritz)
        out = [torch.full((n,), float("nan"), dtype=torch.float64, device="cuda") for _ in range(2)]
        prepared.append((dtype, H, V, ritz, want, out, H.clone(), V.clone()))
    # set-up call: resolves the array's address on this device (and loads its module); from here on nothing allocates
    pkg.chase_residuals_static(prepared[0][1], prepared[0][2], prepared[0][3], prepared[0][5][0])
    torch.cuda.synchronize()
    prepared[0][5][0].fill_(float("nan"))
    free_before = torch.cuda.mem_get_info()[0]
    torch_before = torch.cuda.memory_allocated()
    for dtype, H, V, ritz, want, out, H0, V0 in prepared:
        pkg.chase_residuals_static(H, V, ritz, out[0])          # two calls in a row, same stream
        pkg.chase_residuals_static(H, V, ritz, out[1])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before           # the driver handed out nothing
    assert torch.cuda.memory_allocated() == torch_before         # neither did torch's pool (the wrapper makes no tensor)
    for dtype, H, V, ritz, want, out, H0, V0 in prepared:
        tol = 1e-12 if dtype in (torch.complex128, torch.float64) else 1e-4
        for got in out:
            np.testing.assert_allclose(got.cpu().numpy(), want.cpu().numpy(), rtol=10 * tol)
        assert torch.equal(H, H0) and torch.equal(V, V0)

    # too large for the array: refused, nothing launched, resid untouched
    N, n = 4096, 448
    H = _dev(W.hermitian_gaussian_ensemble(N, torch.complex128, seed=390))
    V = _dev(W.gaussian_colmajor(N, n, torch.complex128, seed=391))
    resid = torch.full((n,), -1.0, dtype=torch.float64, device="cuda")
    launches = pkg.chase_filter_launch_count()
    with pytest.raises(pkg.ChaseFilterError) as ei:
        pkg.chase_residuals_static(H, V, np.zeros(n), resid)
    assert ei.value.code == -8 and pkg.chase_filter_launch_count() == launches
    torch.cuda.synchronize()
    assert bool((resid == -1.0).all())
