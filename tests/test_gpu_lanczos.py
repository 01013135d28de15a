"""GPU parity for Alg. 6: chase_lanczos (coalesced Lanczos runs on the step kernels)
against the NumPy oracle on the same seeded inputs, and the resulting spectral estimates."""
import numpy as np
import pytest
import torch

import paper_1805_10121_b200 as pkg
from oracle import lanczos as OL
from paper_1805_10121_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL = {torch.complex128: 1e-10, torch.float64: 1e-10, torch.complex64: 2e-4, torch.float32: 2e-4}


def _dev(x):
    out = W.empty_colmajor(x.shape[0], x.shape[1], x.dtype, torch.device("cuda:0"))
    out.copy_(x)
    return out


@pytest.mark.parametrize("dtype,N", [(torch.complex128, 1024), (torch.complex128, 520), (torch.float64, 1040),
                                     (torch.complex128, 203), (torch.float64, 301),
                                     (torch.complex64, 768), (torch.float32, 512)])
@pytest.mark.parametrize("k,nruns", [(25, 5), (12, 1)])
def test_lanczos_coefficients_match_oracle(dtype, N, k, nruns):
    w = W.make_config(2, N=N, ncols=nruns, dtype=dtype)
    H, V0 = _dev(w.H), _dev(w.V0)
    alpha, beta = pkg.chase_lanczos(H, V0, k)
    Hn, Vn = w.H.numpy(), w.V0.numpy()
    tol = TOL[dtype]
    for r in range(nruns):
        a_ref, b_ref, _, _ = OL.lanczos(Hn, Vn[:, r], k)
        assert np.max(np.abs(alpha[r] - a_ref)) <= tol * max(1.0, np.max(np.abs(a_ref))), r
        assert np.max(np.abs(beta[r] - b_ref)) <= tol * max(1.0, np.max(np.abs(b_ref))), r
    # inputs untouched
    assert torch.equal(V0.cpu(), w.V0) and torch.equal(H.cpu(), w.H)


def test_spectral_estimates_end_to_end_cfg2_shape():
    """GUE N = 2048: estimates from the GPU Lanczos equal the oracle's, bound the true spectrum
    (eigvalsh) and give usable filter bounds lambda1 < a < b."""
    N, k, nvec, ne = 2048, 25, 4, 128
    w = W.make_config(2, N=N, ncols=1 + nvec)
    alpha, beta = pkg.chase_lanczos(_dev(w.H), _dev(w.V0), k)
    b_sup, mu1, mune = pkg.chase_spectral_estimates(alpha, beta, N, ne)
    Hn, Vn = w.H.numpy(), w.V0.numpy()
    runs = [OL.lanczos(Hn, Vn[:, r], k)[:2] for r in range(1 + nvec)]
    ref = OL.spectral_estimates([r[0] for r in runs], [r[1] for r in runs], N, ne)
    for g, r in zip((b_sup, mu1, mune), ref):
        assert abs(g - r) <= 1e-9
    lam = np.linalg.eigvalsh(Hn)
    assert lam[-1] <= b_sup
    assert lam[0] <= mu1 + 1e-12 and mu1 < mune < b_sup
    assert abs(mune - lam[ne - 1]) <= 0.3


@pytest.mark.parametrize("dtype,N", [(torch.complex128, 520), (torch.float64, 1040), (torch.complex64, 768)])
def test_ritz_vectors_match_oracle_and_land_in_the_chosen_columns(dtype, N):
    """Alg. 6 l.13: Ritz vectors of run 1 below mu_ne, interspersed into every other column of V^; the
    other columns of V^ stay untouched; values and vectors equal the oracle's (unique sign)."""
    k, nruns = 16, 3
    w = W.make_config(2, N=N, ncols=nruns, dtype=dtype)
    H, V0 = _dev(w.H), _dev(w.V0)
    ws = torch.empty(pkg.chase_lanczos_workspace_bytes(N, nruns, k, dtype), dtype=torch.uint8, device="cuda:0")
    alpha, beta = pkg.chase_lanczos(H, V0, k, workspace=ws)
    mu_ne = -0.5
    Vhat0 = W.gaussian_colmajor(N, 2 * k, dtype, seed=99)
    Vhat = _dev(Vhat0)
    dst = list(range(1, 2 * k, 2))                          # odd columns: interspersed with the random ones
    torch.cuda.synchronize()
    # on a non-blocking side stream and with NO synchronisation of ours afterwards: the call itself promises that
    # Vhat is complete on return (the read below runs on the default stream, which does not wait for `side`)
    side = torch.cuda.Stream()
    vals = pkg.chase_lanczos_ritz_vectors(ws, N, dtype, alpha, beta, 1, mu_ne, Vhat, dst, stream=side)
    got = Vhat.cpu().numpy()
    Hn, Vn = w.H.numpy(), w.V0.numpy()
    a_ref, b_ref, U_ref, _ = OL.lanczos(Hn, Vn[:, 1], k)
    lam_ref, X_ref, _ = OL.ritz_vectors(U_ref, a_ref, b_ref, mu_ne)
    assert 0 < len(lam_ref) < k and len(vals) == len(lam_ref)
    tol = 1e-9 if dtype in (torch.complex128, torch.float64) else 2e-3
    np.testing.assert_allclose(vals, lam_ref, atol=tol)
    for i in range(len(vals)):
        assert np.linalg.norm(got[:, dst[i]] - X_ref[:, i]) <= tol * 10, i
    untouched = [c for c in range(2 * k) if c not in dst[: len(vals)]]
    assert np.array_equal(got[:, untouched], Vhat0.numpy()[:, untouched])
    # fewer target columns than Ritz vectors: the smallest Ritz values win
    vals2 = pkg.chase_lanczos_ritz_vectors(ws, N, dtype, alpha, beta, 1, mu_ne, Vhat, dst[:2])
    np.testing.assert_allclose(vals2, lam_ref[:2], atol=tol)
