"""ORACLE -- TEST INFRASTRUCTURE ONLY.  Spectral estimates of ChASE (Alg. 6
"Lanczos procedure for parameters estimates"; Eq. (9)-(10)), in plain NumPy
FP64, step by step in the paper's notation.  Imports nothing from the product package; allowed
callers are tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg.

What the paper fixes and what it leaves open (readings G19-G22):
  * "k Lanczos steps":  A U = U T_k + f_k e_k^T  (Alg. 6 l.2 / l.8).  In exact arithmetic T_k is
    unique given the start vector, whatever variant of the recurrence is used.  The paper mentions
    an "orthogonalization cost" without naming the scheme; reading G19: every new
    vector is orthogonalised against ALL previous Lanczos vectors by two passes of classical
    Gram-Schmidt, alpha_j being the j-th coefficient of the first pass.
  * b_sup = ||f_k||_2 + max(lambda~_1..lambda~_k)                      (Alg. 6 l.3)
  * DoS  phi~(t) = 1/n_vec sum_j sum_i (Z^[j]_{1,i})^2 g_sigma(t - lambda~^[j]_i)   (Eq. 10, l.10)
    with g_sigma the Gaussian density of standard deviation sigma on the eigenvalue axis (G20).
  * mu_{nev+nex} = t-bar with  int_{-inf}^{t-bar} phi~ = (nev+nex)/N   (l.11); "approximately" in the
    paper, here the exact root of the smooth, strictly increasing integral (G21).
  * mu_1 = min_j lambda~^[j]_1                                         (l.12)
  * l.13: "Z^[1] Q^[1]" are the approximate eigenvectors of A; Q^[1] is read as the
    Lanczos basis U^[1] of the first DoS run (the paper's only other use of the letter; reading G22), so
    the i-th Ritz vector is x_i = U^[1] z_i with z_i the eigenvector of T_k for lambda~_i.  Those with
    lambda~_i < mu_{nev+nex} are returned, ascending; WHERE they go in V^ ("intersperse") is the caller's.
The random start vectors are INPUTS (the method's random draws are passed in).
"""
from __future__ import annotations

import math

import numpy as np


def lanczos(H: np.ndarray, v0: np.ndarray, k: int):
    """k Lanczos steps on Hermitian H from the start vector v0 (need not be normalised).

    Returns (alpha[k], beta[k], U[N, k], f[N]) with  H U = U T_k + f e_k^T,
    T_k = tridiag(beta[0..k-2]; alpha[0..k-1]; beta[0..k-2]) and beta[k-1] = ||f||_2.
    """
    H = np.asarray(H)
    wide = np.complex128 if np.iscomplexobj(H) else np.float64
    A = H.astype(wide)
    N = A.shape[0]
    U = np.zeros((N, k), dtype=wide)
    alpha = np.zeros(k)
    beta = np.zeros(k)
    u = np.asarray(v0, dtype=wide).copy()
    u /= np.linalg.norm(u)
    for j in range(k):
        U[:, j] = u
        w = A @ u                                        # one column of the HEMM
        Uj = U[:, : j + 1]
        h = Uj.conj().T @ w                              # first Gram-Schmidt pass (all previous vectors)
        alpha[j] = h[j].real                             # T_k[j, j]
        w = w - Uj @ h
        h2 = Uj.conj().T @ w                             # second pass (re-orthogonalisation)
        w = w - Uj @ h2
        beta[j] = np.linalg.norm(w)                      # T_k[j+1, j]; for j = k-1 this is ||f_k||_2
        if j + 1 < k:
            u = w / beta[j]
    return alpha, beta, U, w


def ritz(alpha: np.ndarray, beta: np.ndarray):
    """T_k = Z^H Lambda~ Z: Ritz values (ascending) and the squared first components (Z_{1,i})^2."""
    k = len(alpha)
    T = np.diag(np.asarray(alpha, dtype=np.float64))
    for j in range(k - 1):
        T[j, j + 1] = T[j + 1, j] = beta[j]
    lam, Z = np.linalg.eigh(T)
    return lam, Z[0, :] ** 2


def ritz_vectors(U: np.ndarray, alpha: np.ndarray, beta: np.ndarray, mu_ne: float):
    """Alg. 6 l.13: Ritz pairs (lam~_i, x_i = U z_i) of one Lanczos run with
    lam~_i < mu_ne, ascending in lam~_i.  T_k z_i = lam~_i z_i by the dense symmetric eigensolver; the
    sign of z_i is fixed by a non-negative first component (it is never zero for beta_j > 0).
    Returns (lam [m], X [N, m], last components |Z_{k,i}| [m])."""
    k = len(alpha)
    T = np.diag(np.asarray(alpha, dtype=np.float64))
    for j in range(k - 1):
        T[j, j + 1] = T[j + 1, j] = beta[j]
    lam, Z = np.linalg.eigh(T)                       # columns of Z: eigenvectors, lam ascending
    Z = Z * np.where(Z[0, :] < 0.0, -1.0, 1.0)[None, :]
    sel = np.nonzero(lam < mu_ne)[0]
    return lam[sel], U @ Z[:, sel], np.abs(Z[k - 1, sel])


def normal_cdf(x: float) -> float:
    return 0.5 * math.erfc(-x / math.sqrt(2.0))


def dos_integral(t: float, lams, weights, sigma: float) -> float:
    """int_{-inf}^{t} phi~(s) ds for phi~ of Eq. (10): lams[j], weights[j] are the Ritz values and
    (Z_{1,i})^2 of run j; the integral of g_sigma(s - lam) up to t is the normal CDF."""
    total = 0.0
    for lam, wts in zip(lams, weights):
        for l, w in zip(lam, wts):
            total += w * normal_cdf((t - l) / sigma)
    return total / len(lams)


def spectral_estimates(alphas, betas, N: int, nev_nex: int, sigma: float = 0.25):
    """Alg. 6 from the Lanczos coefficients of 1 + n_vec runs (run 0: l.2-3; runs 1..n_vec: l.7-8).
    Returns (b_sup, mu_1, mu_nev_nex); with a single run (the `approx` branch, l.4-5) the last two
    are None."""
    lam0, _ = ritz(alphas[0], betas[0])
    b_sup = betas[0][-1] + lam0.max()                                        # l.3
    if len(alphas) == 1:
        return b_sup, None, None                                             # l.4-5
    lams, weights = [], []
    for a, b in zip(alphas[1:], betas[1:]):                                  # l.7-8
        lam, w = ritz(a, b)
        lams.append(lam)
        weights.append(w)
    target = nev_nex / N                                                     # l.11
    lo = min(l.min() for l in lams) - 12.0 * sigma
    hi = max(l.max() for l in lams) + 12.0 * sigma
    for _ in range(200):                                                     # bisection on the integral
        mid = 0.5 * (lo + hi)
        if dos_integral(mid, lams, weights, sigma) < target:
            lo = mid
        else:
            hi = mid
    mu_ne = 0.5 * (lo + hi)
    mu_1 = min(l[0] for l in lams)                                           # l.12
    return b_sup, mu_1, mu_ne
