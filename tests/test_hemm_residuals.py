"""HEMM reuse: chase_hemm (Rayleigh-Ritz's A Q^, Alg. 2 l.2) and
chase_residuals (Alg. 1 l.8) on the filter's step kernels.
CPU part: pins of the oracle (NumPy matmul definition; exact eigenpairs have zero residual; a
two-eigenvector mixture has the closed-form residual eps |lam_j - lam_i| / sqrt(1 + eps^2)).
GPU part: parity of the CUDA path vs the oracle."""
import numpy as np
import pytest
import torch

import oracle
import paper_1805_10121_b200 as pkg
from paper_1805_10121_b200 import workloads as W
from cheb_closed_form import rel_fro


@pytest.mark.parametrize("dtype", [torch.complex128, torch.float64, torch.complex64])
def test_oracle_hemm_vs_numpy_definition(dtype):
    N, n = 130, 9
    H = W.hermitian_gaussian_ensemble(N, dtype, seed=61).numpy()
    X = W.gaussian_colmajor(N, n, dtype, seed=62).numpy()
    Y = W.gaussian_colmajor(N, n, dtype, seed=63).numpy()
    wide = np.complex128 if dtype.is_complex else np.float64
    Hw, Xw, Yw = H.astype(wide), X.astype(wide), Y.astype(wide)
    sh = np.linspace(-1, 1, n)
    got = oracle.hemm(H, X, Y, alpha=0.7, beta=-1.3, shift=sh)
    assert rel_fro(got, 0.7 * (Hw @ Xw - Xw * sh) - 1.3 * Yw) < 1e-14
    got = oracle.hemm(H, X, None, 1.0, 0.0, 0.0)
    assert rel_fro(got, Hw @ Xw) < 1e-14


def test_oracle_residuals_closed_forms():
    N = 120
    H, lam, Q = W.known_spectrum_hermitian(N, torch.complex128, seed=64)
    Hn, lam, Q = H.numpy(), lam.numpy().astype(np.float64), Q.numpy()
    # exact eigenpairs: residual at rounding level
    r = oracle.residuals(Hn, Q[:, :7], lam[:7])
    assert np.all(r < 1e-13)
    # v = (x_i + eps x_j)/sqrt(1+eps^2) with Ritz value lam_i: residual = eps |lam_j - lam_i| / sqrt(1+eps^2)
    i, j, eps = 3, 50, 1e-3
    v = (Q[:, i] + eps * Q[:, j]) / np.sqrt(1 + eps * eps)
    r = oracle.residuals(Hn, v[:, None], [lam[i]])
    assert r[0] == pytest.approx(eps * abs(lam[j] - lam[i]) / np.sqrt(1 + eps * eps), rel=1e-9)


def _dev(x):
    out = W.empty_colmajor(x.shape[0], x.shape[1], x.dtype, "cuda")
    out.copy_(x)
    return out


@pytest.mark.gpu
@pytest.mark.parametrize("dtype,N,n", [(torch.complex128, 520, 77), (torch.float64, 1040, 150),
                                        (torch.complex64, 300, 33), (torch.float32, 203, 20), (torch.float32, 516, 70),
                                        (torch.complex64, 1282, 140),
                                        (torch.complex128, 203, 20)])
def test_gpu_hemm_and_residuals(dtype, N, n):
    tol = 1e-12 if dtype in (torch.complex128, torch.float64) else 1e-4
    H = W.hermitian_gaussian_ensemble(N, dtype, seed=71)
    X = W.gaussian_colmajor(N, n, dtype, seed=72)
    Y = W.gaussian_colmajor(N, n, dtype, seed=73)
    Hd, Xd, Yd = _dev(H), _dev(X), _dev(Y)
    pkg.chase_hemm(Hd, Xd, Yd, alpha=0.7, beta=-1.3, shift=0.25)
    ref = oracle.hemm(H.numpy(), X.numpy(), Y.numpy(), 0.7, -1.3, 0.25)
    assert rel_fro(Yd.cpu().numpy(), ref) <= tol
    Yd.fill_(float("nan"))                       # beta = 0: Y must not be read
    pkg.chase_hemm(Hd, Xd, Yd)
    assert rel_fro(Yd.cpu().numpy(), oracle.hemm(H.numpy(), X.numpy(), None)) <= tol
    ritz = np.linspace(-2, 2, n)
    got = pkg.chase_residuals(Hd, Xd, ritz).cpu().numpy()
    ref = oracle.residuals(H.numpy(), X.numpy(), ritz)
    np.testing.assert_allclose(got, ref, rtol=10 * tol)
    assert torch.equal(Xd.cpu(), X)              # V is read-only


@pytest.mark.gpu
def test_gpu_residuals_of_exact_eigenpairs():
    w = W.make_config(1)
    Q = W.as_colmajor(w.eigvecs[:, :40].contiguous())
    r = pkg.chase_residuals(_dev(w.H), _dev(Q), w.eigvals[:40].numpy().astype(np.float64)).cpu().numpy()
    assert np.all(r < 1e-13)


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", [torch.float32, torch.float64, torch.complex64, torch.complex128])
@pytest.mark.parametrize("N,n", [(1040, 5), (203, 1), (777, 8), (1536, 3), (64, 7), (2600, 2), (4100, 6), (130, 4)])
def test_gpu_skinny_hemm_and_residuals(dtype, N, n):
    """1..8 columns take the streaming kernels (csrc/step_stream.cu: bulk-copy ring, when the columns of
    H start on 16-byte boundaries; csrc/step_skinny.cu otherwise): all dtypes, odd N, several persistent
    column blocks per CTA, ragged last block and last stage, beta = 0 must not read Y, per-column shifts
    (residuals)."""
    tol = 1e-12 if dtype in (torch.complex128, torch.float64) else 2e-5
    H = W.hermitian_gaussian_ensemble(N, dtype, seed=91)
    X = W.gaussian_colmajor(N, n, dtype, seed=92)
    Y = W.gaussian_colmajor(N, n, dtype, seed=93)
    Hd, Xd, Yd = _dev(H), _dev(X), _dev(Y)
    pkg.chase_hemm(Hd, Xd, Yd, alpha=0.7, beta=-1.3, shift=0.25)
    assert rel_fro(Yd.cpu().numpy(), oracle.hemm(H.numpy(), X.numpy(), Y.numpy(), 0.7, -1.3, 0.25)) <= tol
    Yd.fill_(float("nan"))
    pkg.chase_hemm(Hd, Xd, Yd)
    assert rel_fro(Yd.cpu().numpy(), oracle.hemm(H.numpy(), X.numpy(), None)) <= tol
    ritz = np.linspace(-2, 2, n)
    got = pkg.chase_residuals(Hd, Xd, ritz).cpu().numpy()
    np.testing.assert_allclose(got, oracle.residuals(H.numpy(), X.numpy(), ritz), rtol=10 * tol)
    assert torch.equal(Xd.cpu(), X) and torch.equal(Hd.cpu(), H)


@pytest.mark.gpu
@pytest.mark.parametrize("dtype,N,n", [(torch.complex128, 520, 77), (torch.float64, 1040, 150)])
def test_gpu_hemm_on_side_stream_with_cold_scratch_cache(dtype, N, n):
    """chase_hemm brings no workspace: on the FP64 tensor path its stream-K flags live in a cached buffer the
    library allocates on first use.  That buffer must be zeroed on the LAUNCHING stream -- a non-blocking
    side stream does not wait for the legacy default stream -- so: empty the cache, launch on a fresh
    torch stream, several times over."""
    H = W.hermitian_gaussian_ensemble(N, dtype, seed=75)
    X = W.gaussian_colmajor(N, n, dtype, seed=76)
    Hd, Xd = _dev(H), _dev(X)
    ref = oracle.hemm(H.numpy(), X.numpy(), None)
    torch.cuda.synchronize()
    for _ in range(4):
        pkg.chase_scratch_cache_release()
        st = torch.cuda.Stream()
        Yd = W.empty_colmajor(N, n, dtype, "cuda")
        Yd.fill_(float("nan"))
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            pkg.chase_hemm(Hd, Xd, Yd, stream=st)
            pkg.chase_hemm(Hd, Xd, Yd, alpha=1.0, beta=0.0, stream=st)      # warm slot, next epoch
        st.synchronize()
        assert rel_fro(Yd.cpu().numpy(), ref) <= 1e-12
    pkg.chase_scratch_cache_release()
    pkg.chase_scratch_cache_release()                                        # empty cache: a no-op
