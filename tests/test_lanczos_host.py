"""CPU-only: chase_spectral_estimates (host side of Alg. 6) against the oracle on
Lanczos coefficients produced by the oracle, plus its argument validation."""
import math

import numpy as np
import pytest

import paper_1805_10121_b200 as pkg
from oracle import lanczos as OL


def _coeffs(N, k, nruns, seed, cplx=True):
    rng = np.random.default_rng(seed)
    G = rng.standard_normal((N, N)) + (1j * rng.standard_normal((N, N)) if cplx else 0)
    H = (G + G.conj().T) / math.sqrt(2 * N * (2 if cplx else 1))
    runs = [OL.lanczos(H, rng.standard_normal(N) + 0j, k)[:2] for _ in range(nruns)]
    return np.array([r[0] for r in runs]), np.array([r[1] for r in runs])


@pytest.mark.parametrize("N,k,nruns,ne,sigma", [(300, 25, 5, 40, 0.25), (200, 12, 5, 20, 0.25),
                                                (150, 40, 11, 75.5, 0.1), (64, 64, 3, 10, 0.05)])
def test_estimates_match_oracle(N, k, nruns, ne, sigma):
    al, be = _coeffs(N, k, nruns, 7 + k)
    ref = OL.spectral_estimates(list(al), list(be), N, ne, sigma)
    got = pkg.chase_spectral_estimates(al, be, N, ne, sigma)
    for g, r in zip(got, ref):
        assert abs(g - r) <= 1e-11 * max(1.0, abs(r))


def test_approx_branch_returns_only_b_sup():
    al, be = _coeffs(100, 10, 1, 3)
    b_sup, mu1, mune = pkg.chase_spectral_estimates(al, be, 100, 10)
    lam, _ = OL.ritz(al[0], be[0])
    assert mu1 is None and mune is None
    assert abs(b_sup - (be[0][-1] + lam.max())) <= 1e-13


def test_ritz_weights_via_single_gaussian_limit():
    """With ONE DoS run and a very wide kernel the integral is ~ Phi((t - mean)/sigma) with
    mean = sum_i w_i lam_i = alpha_0 (first Gauss moment), so t-bar at 1/2 is alpha[1][0]."""
    al, be = _coeffs(120, 8, 2, 5)
    sigma = 1e4
    _, _, mune = pkg.chase_spectral_estimates(al, be, 120, 60, sigma)
    assert abs(mune - al[1][0]) <= 1e-3


def test_validation():
    al, be = _coeffs(50, 6, 3, 1)
    E = pkg.ChaseFilterError
    with pytest.raises(E):
        pkg.chase_spectral_estimates(al, be, 50, 10, sigma=0.0)
    with pytest.raises(E):
        pkg.chase_spectral_estimates(al, be, 50, 50, sigma=0.25)      # nev_nex must be < N
    with pytest.raises(E):
        pkg.chase_spectral_estimates(al, be, 50, 0, sigma=0.25)
    bad = be.copy(); bad[1, 2] = float("nan")
    with pytest.raises(E):
        pkg.chase_spectral_estimates(al, bad, 50, 10)
    assert pkg.chase_lanczos_workspace_bytes(0, 5, 25, __import__("torch").float64) == 0
    assert pkg.chase_lanczos_workspace_bytes(100, 5, 25, __import__("torch").complex128) >= 100 * 5 * 26 * 16


def test_ritz_vectors_reject_duplicate_destination_columns():
    """Two Ritz vectors aimed at one column of V^ would race in the kernel: refused before any CUDA call
    (fake device pointers, never dereferenced)."""
    import numpy as np
    lib = pkg.load()
    k, nruns, N = 6, 2, 64
    al, be = _coeffs(N, k, nruns, 1)
    al, be = np.ascontiguousarray(al), np.ascontiguousarray(be)
    cnt = np.zeros(1, dtype=np.int64)
    wsb = pkg.chase_lanczos_workspace_bytes(N, nruns, k, __import__("torch").float64)

    def call(dst):
        d = np.asarray(dst, dtype=np.int64)
        return lib.chase_lanczos_ritz_vectors(0x1000, wsb, N, nruns, k, 1, 1, al.ctypes.data, be.ctypes.data, -1e9,
                                              0x2000, 8, d.ctypes.data, d.size, cnt.ctypes.data, None, None)

    assert call([1, 3, 1]) == -1
    assert call([1, 3, 8]) == -1                 # out of range
    assert call([1, 3, 5]) == 0 and cnt[0] == 0  # mu_ne below every Ritz value: nothing written, nothing launched
