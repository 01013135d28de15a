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
