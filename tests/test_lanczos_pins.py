"""Pins for the Lanczos / DoS oracle (oracle/lanczos.py; Alg. 6, Eq. 9-10) against
what the mathematics fixes: the Lanczos relation and orthogonality, Gauss-quadrature exactness of
(Ritz values, (Z_1i)^2), the k = N limit, the b_sup bound on known spectra, and the DoS integral
against a direct quadrature of Eq. (10).  CPU only."""
import math

import numpy as np
import pytest

from oracle import lanczos as OL


def _hermitian(N, seed, cplx=True):
    rng = np.random.default_rng(seed)
    G = rng.standard_normal((N, N)) + (1j * rng.standard_normal((N, N)) if cplx else 0)
    H = (G + G.conj().T) / math.sqrt(2 * N * (2 if cplx else 1))
    return H


def _known_spectrum(N, lam, seed):
    rng = np.random.default_rng(seed)
    Q, _ = np.linalg.qr(rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N)))
    H = (Q * lam) @ Q.conj().T
    return (H + H.conj().T) / 2, Q


@pytest.mark.parametrize("cplx", [True, False])
def test_L1_lanczos_relation_and_orthogonality(cplx):
    """A U = U T_k + f e_k^T (Alg. 6 l.2), U^H U = I, U^H f = 0."""
    N, k = 300, 25
    H = _hermitian(N, 1, cplx)
    v0 = np.random.default_rng(2).standard_normal(N) + (1j if cplx else 0) * np.random.default_rng(3).standard_normal(N)
    alpha, beta, U, f = OL.lanczos(H, v0, k)
    T = np.diag(alpha) + np.diag(beta[:-1], 1) + np.diag(beta[:-1], -1)
    R = H @ U - U @ T
    R[:, -1] -= f
    assert np.linalg.norm(R) <= 1e-13 * np.linalg.norm(H)
    assert np.linalg.norm(U.conj().T @ U - np.eye(k)) <= 1e-13
    assert np.linalg.norm(U.conj().T @ f) <= 1e-13
    assert abs(np.linalg.norm(f) - beta[-1]) <= 1e-15
    assert np.allclose(U[:, 0], v0 / np.linalg.norm(v0))
    assert np.all(beta > 0)


def test_L2_gauss_quadrature_moments():
    """(Ritz values, (Z_1i)^2) of k Lanczos steps are the k-point Gauss rule of the spectral measure of
    v0: sum_i w_i lam_i^p = v^H A^p v / v^H v for every p <= 2k-1 -- and NOT for p = 2k."""
    N, k = 120, 6
    lam_true = np.linspace(-1.0, 1.5, N)
    H, _ = _known_spectrum(N, lam_true, 5)
    v0 = np.random.default_rng(6).standard_normal(N) + 1j * np.random.default_rng(7).standard_normal(N)
    alpha, beta, _, _ = OL.lanczos(H, v0, k)
    lam, w = OL.ritz(alpha, beta)
    assert abs(w.sum() - 1.0) <= 1e-14
    v = v0 / np.linalg.norm(v0)
    x = v.copy()
    for p in range(2 * k + 1):
        exact = np.vdot(v, x).real                  # v^H A^p v
        quad = float(np.sum(w * lam ** p))
        if p <= 2 * k - 1:
            assert abs(quad - exact) <= 1e-12 * max(1.0, abs(exact)), p
        else:
            assert abs(quad - exact) > 1e-9          # degree 2k is the first the rule misses
        x = H @ x


def test_L3_full_krylov_space_recovers_the_spectrum():
    """k = N: T_N is unitarily similar to A, Ritz values = eigenvalues, weights = |q_i^H v|^2, f = 0."""
    N = 24
    lam_true = np.sort(np.random.default_rng(8).uniform(-1, 1, N))
    H, Q = _known_spectrum(N, lam_true, 9)
    v0 = np.random.default_rng(10).standard_normal(N) + 0j
    alpha, beta, _, f = OL.lanczos(H, v0, N)
    lam, w = OL.ritz(alpha, beta)
    assert np.allclose(lam, lam_true, atol=1e-10)
    coef = np.abs(Q.conj().T @ (v0 / np.linalg.norm(v0))) ** 2
    assert np.allclose(w, coef, atol=1e-8)
    assert np.linalg.norm(f) <= 1e-8


@pytest.mark.parametrize("seed", [11, 12, 13, 14])
def test_L4_b_sup_is_an_upper_bound(seed):
    """b_sup = ||f_k|| + max Ritz value (Alg. 6 l.3) must bound the spectrum and not be
    absurdly loose (|b_sup - lam_max| <= ||f_k||)."""
    N, k = 400, 25
    H = _hermitian(N, seed)
    lam_max = np.linalg.eigvalsh(H)[-1]
    v0 = np.random.default_rng(seed + 100).standard_normal(N) + 0j
    alpha, beta, _, _ = OL.lanczos(H, v0, k)
    b_sup, mu1, mune = OL.spectral_estimates([alpha], [beta], N, 40)
    assert mu1 is None and mune is None                # the `approx` branch, l.4-5
    assert lam_max <= b_sup <= lam_max + beta[-1] + 1e-12


def test_L5_dos_integral_matches_direct_quadrature_of_eq10():
    """int phi~ from -inf to t-bar, phi~ written out as Eq. (10) with the Gaussian density
    exp(-x^2 / 2 sigma^2) / sqrt(2 pi sigma^2) and integrated by the trapezoid rule, equals
    (nev+nex)/N at the returned mu_{nev+nex}; total mass 1."""
    N, k, nvec, sigma = 500, 25, 4, 0.25
    H = _hermitian(N, 21)
    rng = np.random.default_rng(22)
    runs = [OL.lanczos(H, rng.standard_normal(N) + 1j * rng.standard_normal(N), k)[:2] for _ in range(1 + nvec)]
    alphas, betas = [r[0] for r in runs], [r[1] for r in runs]
    nev_nex = 60
    b_sup, mu1, mune = OL.spectral_estimates(alphas, betas, N, nev_nex, sigma)
    lw = [OL.ritz(a, b) for a, b in zip(alphas[1:], betas[1:])]

    def phi(t):
        s = 0.0
        for lam, w in lw:
            s = s + np.sum(w[None, :] * np.exp(-(t[:, None] - lam[None, :]) ** 2 / (2 * sigma ** 2)), axis=1)
        return s / (nvec * math.sqrt(2 * math.pi * sigma ** 2))

    def trapezoid(y, x):
        return float(np.sum(0.5 * (y[1:] + y[:-1]) * np.diff(x)))

    t = np.linspace(-8.0, mune, 200001)
    assert abs(trapezoid(phi(t), t) - nev_nex / N) <= 1e-8
    t = np.linspace(-8.0, 8.0, 200001)
    assert abs(trapezoid(phi(t), t) - 1.0) <= 1e-8
    assert mu1 == min(l[0] for l, _ in lw)                                   # l.12
    assert mu1 < mune < b_sup


def test_L6_diagonal_matrix_quantile():
    """A = diag(h), v0 = ones, k = N: weights 1/N, Ritz values h, so phi~ is Eq. (9) itself and with a
    narrow kernel t-bar is the (nev+nex)/N quantile: it lies between h_(m) and h_(m+1)."""
    N, m = 40, 10
    h = np.sort(np.random.default_rng(31).uniform(-2, 2, N))
    H = np.diag(h)
    alpha, beta, _, _ = OL.lanczos(H, np.ones(N), N)
    lam, w = OL.ritz(alpha, beta)
    assert np.allclose(lam, h, atol=1e-9) and np.allclose(w, 1.0 / N, atol=1e-7)
    gap = np.min(np.diff(h))
    _, mu1, mune = OL.spectral_estimates([alpha, alpha], [beta, beta], N, m + 0.5, sigma=gap / 20)
    assert h[m - 1] < mune < h[m] + gap
    assert abs(mu1 - h[0]) <= 1e-9


def test_L7_gue_estimates_are_sane():
    """GUE N = 1000: true spectrum from eigvalsh.  mu_1 is a Ritz value (>= lam_min, and close), b_sup a
    bound, mu_{nev+nex} within the kernel width of the true (nev+nex)-th eigenvalue."""
    N, k, nvec, nev_nex = 1000, 25, 4, 60
    H = _hermitian(N, 41)
    lam_true = np.linalg.eigvalsh(H)
    rng = np.random.default_rng(42)
    runs = [OL.lanczos(H, rng.standard_normal(N) + 1j * rng.standard_normal(N), k)[:2] for _ in range(1 + nvec)]
    b_sup, mu1, mune = OL.spectral_estimates([r[0] for r in runs], [r[1] for r in runs], N, nev_nex, 0.25)
    assert lam_true[-1] <= b_sup <= lam_true[-1] + runs[0][1][-1] + 1e-12   # loose by at most ||f_k|| (~1 for GUE)
    assert lam_true[0] - 1e-12 <= mu1 <= lam_true[0] + 0.1
    assert abs(mune - lam_true[nev_nex - 1]) <= 0.3


def test_l8_ritz_vectors_residual_identity_and_orthonormality():
    """Alg. 6 l.13.  Pins oracle.lanczos.ritz_vectors with what the mathematics fixes:
    the classical Lanczos residual identity  ||A x_i - lam~_i x_i||_2 = beta_k |Z_{k,i}|  (from
    A U = U T + f e_k^T, ||f|| = beta_k), orthonormality of the x_i, Rayleigh quotients x_i^H A x_i = lam~_i,
    the selection lam~_i < mu_ne in ascending order, and -- for k = N, where the Krylov space is the whole
    space -- that the Ritz pairs ARE the eigenpairs of A (eigh), up to the fixed sign."""
    rng = np.random.default_rng(77)
    N, k = 120, 14
    G = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    A = (G + G.conj().T) / np.sqrt(2 * N)
    v0 = rng.standard_normal(N) + 1j * rng.standard_normal(N)
    alpha, beta, U, f = OL.lanczos(A, v0, k)
    mu = 0.3
    lam, X, zk = OL.ritz_vectors(U, alpha, beta, mu)
    all_lam, _ = OL.ritz(alpha, beta)
    assert len(lam) == int(np.sum(all_lam < mu)) and 0 < len(lam) < k
    assert np.all(np.diff(lam) > 0) and np.all(lam < mu)
    R = A @ X - X * lam[None, :]
    np.testing.assert_allclose(np.linalg.norm(R, axis=0), beta[-1] * zk, rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(X.conj().T @ X, np.eye(len(lam)), atol=1e-12)
    np.testing.assert_allclose(np.real(np.einsum("ij,ij->j", X.conj(), A @ X)), lam, atol=1e-12)
    # a wrong index (e.g. Z rows instead of columns) or a transposed operand breaks the identity above;
    # the direction of the residual pins it further: R = f * Z_{k,i} exactly
    Zk_signed = (X.conj().T @ U[:, -1:])[:, 0].conj()      # = Z_{k,i} since x_i = U z_i, U orthonormal
    np.testing.assert_allclose(R, np.outer(f, Zk_signed), atol=1e-10)

    # k = N: Ritz pairs = eigenpairs
    N2 = 24
    A2 = A[:N2, :N2]
    alpha2, beta2, U2, _ = OL.lanczos(A2, v0[:N2], N2)
    lam2, X2, _ = OL.ritz_vectors(U2, alpha2, beta2, np.inf)
    w, Q = np.linalg.eigh(A2)
    np.testing.assert_allclose(lam2, w, atol=1e-10)
    overlap = np.abs(np.einsum("ij,ij->j", Q.conj(), X2))
    np.testing.assert_allclose(overlap, 1.0, atol=1e-8)
