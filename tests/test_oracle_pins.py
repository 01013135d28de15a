"""Pins of the CPU oracle against what the paper and the mathematics fix (-m "not gpu").

P1 spectral closed form, P2 sigma closed form, P3 degree-1 brute force, P4 gain
invariants (Thm 4.2), P5 H = cI / diagonal special cases, P6 reflector closed form,
P7 column independence, P8 linearity, P9 uniform vs mixed degrees.
Citations: PAPER.md:259-262 (Def. 4.1), :266 (Eq. 3), :289-303 (Thm 4.2, Eq. 5),
:311-313 (Eq. 7), :321-350 (Alg. 4).
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1805_10121_b200 import workloads as W
from cheb_closed_form import cheb_C, p_m, rel_fro


def _np(t: torch.Tensor) -> np.ndarray:
    return t.numpy()


@pytest.fixture(scope="module")
def cfg1():
    return W.make_config(1)


def _spectral_closed_form(Q, lam, V0, degrees, a, b, lambda1):
    """Q diag(p_{m_j}(lam)) Q^H V0[:, j], column by column."""
    coef = Q.conj().T @ V0
    out = np.empty_like(coef)
    for j, m in enumerate(degrees):
        out[:, j] = Q @ (p_m(int(m), lam, a, b, lambda1) * coef[:, j])
    return out


# ---- P1 -------------------------------------------------------------------------------
def test_p1_spectral_closed_form_cfg1(cfg1):
    w = cfg1
    out = oracle.chase_filter(_np(w.H), _np(w.V0), _np(w.degrees), w.a, w.b, w.lambda1)
    ref = _spectral_closed_form(_np(w.eigvecs), _np(w.eigvals).astype(np.float64), _np(w.V0),
                                _np(w.degrees), w.a, w.b, w.lambda1)
    assert rel_fro(out, ref) < 1e-12


@pytest.mark.parametrize("dtype", [torch.complex128, torch.float64])
def test_p1_spectral_closed_form_mixed_degrees(dtype):
    """Mixed degrees incl. 0, 1, odd ones (readings G5, G6) on a known-spectrum matrix."""
    N, n = 192, 24
    H, lam, Q = W.known_spectrum_hermitian(N, dtype, seed=11)
    V0 = W.gaussian_colmajor(N, n, dtype, seed=12)
    deg = np.sort(np.array([0, 0, 1, 1, 2, 3, 4, 5, 6, 7, 8, 8, 9, 10, 12, 13, 16, 18, 20, 21, 28, 30, 35, 36],
                           dtype=np.int32))
    a, b, l1 = float(lam[n]), float(lam[-1]) + 0.01, float(lam[0]) - 0.02
    out = oracle.chase_filter(_np(H), _np(V0), deg, a, b, l1)
    ref = _spectral_closed_form(_np(Q), _np(lam).astype(np.float64), _np(V0), deg, a, b, l1)
    assert rel_fro(out, ref) < 1e-11
    for j in range(n):  # per column too: a wrong result in a tiny-norm column must not hide
        assert rel_fro(out[:, j], ref[:, j]) < 1e-10


def test_p1_via_eigh_gue():
    """GUE recipe of cfg 2 at reduced N, closed form through numpy's eigh."""
    w = W.make_config(2, N=384, ncols=32)
    Hn = _np(w.H)
    lam, Q = np.linalg.eigh(Hn)
    out = oracle.chase_filter(Hn, _np(w.V0), _np(w.degrees), w.a, w.b, w.lambda1)
    ref = _spectral_closed_form(Q, lam, _np(w.V0), _np(w.degrees), w.a, w.b, w.lambda1)
    assert rel_fro(out, ref) < 1e-11


# ---- P2 -------------------------------------------------------------------------------
def test_p2_sigma_closed_form():
    a, b, l1 = -1.7, 2.05, -2.0
    m = 36
    sigma, alpha, beta, c, e = oracle.chase_scalars(a, b, l1, m)
    assert c == pytest.approx((a + b) / 2) and e == pytest.approx((b - a) / 2)
    tg = (l1 - c) / e
    assert tg < -1.0
    ks = np.arange(1, m + 1)
    C = np.array([cheb_C(k, np.array([tg]))[0] for k in range(0, m + 1)])
    np.testing.assert_allclose(sigma[1:], C[ks - 1] / C[ks], rtol=1e-13)      # sigma_k = C_{k-1}/C_k
    rho = abs(tg) + np.sqrt(tg * tg - 1.0)
    assert sigma[m] == pytest.approx(-1.0 / rho, rel=1e-6)                    # limit -1/rho_gamma
    d = np.diff(np.abs(sigma[1:]))                                            # |sigma_k| decreasing ...
    assert np.all(d <= 0) and np.all(d[:12] < 0)                              # ... until FP64 saturates
    np.testing.assert_allclose(alpha[1], sigma[1] / e, rtol=1e-15)
    assert beta[1] == 0.0
    np.testing.assert_allclose(alpha[2:], 2 * sigma[2:] / e, rtol=1e-14)      # Eq. (7)
    np.testing.assert_allclose(beta[2:], -sigma[2:] * sigma[1:-1], rtol=1e-14)


def test_p2_recurrence_reproduces_chebyshev_scalars():
    """With scalars alpha_k, beta_k the scalar recurrence y_k = alpha_k (x-c) y_{k-1} + beta_k y_{k-2}
    must give p_k(x) (Eq. 5) for any x: pins alpha/beta jointly (a dropped sigma<-tau fails here)."""
    a, b, l1 = -0.4, 1.3, -1.1
    m = 30
    _, alpha, beta, c, _ = oracle.chase_scalars(a, b, l1, m)
    x = np.linspace(-1.5, 1.3, 57)
    y_prev, y = np.ones_like(x), alpha[1] * (x - c)
    for k in range(2, m + 1):
        y_prev, y = y, alpha[k] * (x - c) * y + beta[k] * y_prev
        np.testing.assert_allclose(y, p_m(k, x, a, b, l1), rtol=1e-10, atol=1e-13)


# ---- P3 -------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", [torch.complex128, torch.float64, torch.complex64, torch.float32])
def test_p3_degree1_brute_force(dtype):
    N, n = 150, 7
    H = W.hermitian_gaussian_ensemble(N, dtype, seed=21)
    V0 = W.gaussian_colmajor(N, n, dtype, seed=22)
    a, b, l1 = -1.5, 2.1, -2.2
    out = oracle.chase_filter(_np(H), _np(V0), np.ones(n, np.int32), a, b, l1)
    c, e = (a + b) / 2, (b - a) / 2
    wide = np.complex128 if dtype.is_complex else np.float64
    Hn, Vn = _np(H).astype(wide), _np(V0).astype(wide)
    ref = (1.0 / (l1 - c)) * (Hn @ Vn - c * Vn)       # (sigma_1/e)(H - cI)V0, sigma_1/e = 1/(lambda1-c)
    assert rel_fro(out, ref) < 1e-14


def test_p3_degree2_brute_force():
    """One full recurrence step by hand (Eq. 7 with m = 1)."""
    N, n = 96, 5
    H = W.hermitian_gaussian_ensemble(N, torch.complex128, seed=23)
    V0 = W.gaussian_colmajor(N, n, torch.complex128, seed=24)
    a, b, l1 = -1.2, 2.2, -2.4
    c, e = (a + b) / 2, (b - a) / 2
    s1 = e / (l1 - c)
    s2 = 1.0 / (2.0 / s1 - s1)
    Hn, Vn = _np(H), _np(V0)
    A = Hn - c * np.eye(N)
    V1 = (s1 / e) * (A @ Vn)
    V2 = (2 * s2 / e) * (A @ V1) - s2 * s1 * Vn
    out = oracle.chase_filter(Hn, Vn, np.full(n, 2, np.int32), a, b, l1)
    assert rel_fro(out, V2) < 1e-14


# ---- P4 -------------------------------------------------------------------------------
def test_p4_gain_invariants(cfg1):
    """Thm 4.2 / Eq. 6: gain exactly 1 at lambda_1; |gain| <= 1/|C_m(t_gamma)| on [a,b];
    gain above that bound and monotone decreasing in lambda below a."""
    w = cfg1
    m = int(w.degrees[0])
    Q, lam = _np(w.eigvecs), _np(w.eigvals).astype(np.float64)
    out = oracle.chase_filter(_np(w.H), _np(w.V0), _np(w.degrees), w.a, w.b, w.lambda1)
    cin = Q.conj().T @ _np(w.V0)
    cout = Q.conj().T @ out
    gain = (cout / cin)                     # per eigen-direction and column
    assert np.max(np.abs(gain.imag)) < 1e-9
    g = gain.real.mean(axis=1)
    assert np.max(np.abs(gain.real - g[:, None])) < 1e-9        # same gain for every column
    c, e = (w.a + w.b) / 2, (w.b - w.a) / 2
    bound = 1.0 / abs(cheb_C(m, np.array([(w.lambda1 - c) / e]))[0])
    assert g[0] == pytest.approx(1.0, abs=1e-12)                # p_m(lambda_1) = 1
    unwanted = lam >= w.a
    wanted = lam < w.a
    assert wanted.sum() == w.ncols
    assert np.all(np.abs(g[unwanted]) <= bound * (1 + 1e-9))
    assert np.all(g[wanted] > bound)
    assert np.all(np.diff(g[wanted]) < 0)                       # monotone: lower lambda, larger gain
    assert g[wanted].min() > np.abs(g[unwanted]).max()


# ---- P5 -------------------------------------------------------------------------------
def test_p5_scalar_matrix():
    """H = c I: V_1 = 0, V_2 = -sigma_1 sigma_2 V_0, and generally V_m = p_m(c) V_0."""
    N, n = 64, 4
    a, b, l1 = -1.0, 3.0, -2.5
    c = (a + b) / 2
    H = np.asfortranarray(np.eye(N) * c)
    V0 = _np(W.gaussian_colmajor(N, n, torch.float64, seed=31))
    deg = np.array([1, 2, 3, 8], np.int32)
    out = oracle.chase_filter(H, V0, deg, a, b, l1)
    assert np.all(out[:, 0] == 0.0)
    e = (b - a) / 2
    s1 = e / (l1 - c)
    s2 = 1 / (2 / s1 - s1)
    np.testing.assert_allclose(out[:, 1], -s1 * s2 * V0[:, 1], rtol=1e-14)
    assert np.all(out[:, 2] == 0.0)                                   # odd polynomial at t = 0
    np.testing.assert_allclose(out[:, 3], p_m(8, np.array([c]), a, b, l1)[0] * V0[:, 3], rtol=1e-12)


@pytest.mark.parametrize("dtype", [torch.complex128, torch.float64])
def test_p5_diagonal_matrix(dtype):
    """H = diag(h): out[i,j] = p_{m_j}(h_i) V0[i,j] element-wise."""
    N, n = 300, 6
    rng = np.random.default_rng(5)
    h = rng.uniform(-2.5, 2.0, N)
    wide = np.complex128 if dtype.is_complex else np.float64
    H = np.asfortranarray(np.diag(h).astype(wide))
    V0 = _np(W.gaussian_colmajor(N, n, dtype, seed=32))
    deg = np.array([2, 4, 10, 20, 30, 36], np.int32)
    a, b, l1 = -1.7, 2.05, -2.0
    out = oracle.chase_filter(H, V0, deg, a, b, l1)
    for j, m in enumerate(deg):
        ref = p_m(int(m), h, a, b, l1) * V0[:, j]
        assert rel_fro(out[:, j], ref) < 1e-11


# ---- P6 -------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", [torch.complex128, torch.float64])
def test_p6_reflector_closed_form(dtype):
    N, n = 700, 9
    H, lam, us = W.reflector_hermitian(N, dtype, seed=41)
    V0 = _np(W.gaussian_colmajor(N, n, dtype, seed=42))
    lam = _np(lam)
    deg = np.array([2, 4, 6, 8, 10, 14, 20, 28, 36], np.int32)
    a, b, l1 = float(lam[n + 20]), 2.01, float(lam[0]) - 1e-3

    def R(x):          # R = R_1 R_2 ...
        for u in reversed(us):
            un = u.numpy()
            x = x - 2.0 * np.outer(un, un.conj() @ x)
        return x

    def RH(x):         # R^H = ... R_2 R_1
        for u in us:
            un = u.numpy()
            x = x - 2.0 * np.outer(un, un.conj() @ x)
        return x

    coef = RH(V0)
    for j, m in enumerate(deg):
        coef[:, j] *= p_m(int(m), lam, a, b, l1)
    ref = R(coef)
    out = oracle.chase_filter(_np(H), V0, deg, a, b, l1)
    assert rel_fro(out, ref) < 1e-11


# ---- P7 / P8 / P9 ---------------------------------------------------------------------
@pytest.fixture(scope="module")
def small_mixed():
    w = W.make_config(2, N=256, ncols=40)
    out = oracle.chase_filter(_np(w.H), _np(w.V0), _np(w.degrees), w.a, w.b, w.lambda1)
    return w, out


def test_p7_column_independence(small_mixed):
    w, out = small_mixed
    cols = np.array([0, 3, 17, 18, 39])
    sub = oracle.chase_filter(_np(w.H), _np(w.V0)[:, cols], _np(w.degrees)[cols], w.a, w.b, w.lambda1)
    assert np.array_equal(sub, out[:, cols])      # same k-ascending sums -> bitwise equal


def test_p8_linearity(small_mixed):
    w, out = small_mixed
    s = np.linspace(0.5, 2.0, w.ncols)
    scaled = oracle.chase_filter(_np(w.H), _np(w.V0) * s, _np(w.degrees), w.a, w.b, w.lambda1)
    assert rel_fro(scaled, out * s) < 1e-14
    deg = np.full(w.ncols // 2, 12, np.int32)
    X, Y = _np(w.V0)[:, :20], _np(w.V0)[:, 20:]
    fx = oracle.chase_filter(_np(w.H), X, deg, w.a, w.b, w.lambda1)
    fy = oracle.chase_filter(_np(w.H), Y, deg, w.a, w.b, w.lambda1)
    fxy = oracle.chase_filter(_np(w.H), X + 2.0 * Y, deg, w.a, w.b, w.lambda1)
    assert rel_fro(fxy, fx + 2.0 * fy) < 1e-13


def test_p9_uniform_vs_mixed_degrees(small_mixed):
    w, out = small_mixed
    deg = _np(w.degrees)
    assert len(np.unique(deg)) > 3
    for d in np.unique(deg):
        cols = np.nonzero(deg == d)[0]
        uni = oracle.chase_filter(_np(w.H), _np(w.V0)[:, cols], np.full(len(cols), d, np.int32),
                                  w.a, w.b, w.lambda1)
        assert np.array_equal(uni, out[:, cols])


# ---- single-precision inputs, degree 0, misc ----------------------------------------------
def test_f32_inputs_are_upcast_exactly():
    w = W.make_config(5, N=128, ncols=8)
    assert w.dtype == torch.complex64
    out32 = oracle.chase_filter(_np(w.H), _np(w.V0), _np(w.degrees), w.a, w.b, w.lambda1)
    out64 = oracle.chase_filter(_np(w.H).astype(np.complex128), _np(w.V0).astype(np.complex128),
                                _np(w.degrees), w.a, w.b, w.lambda1)
    assert out32.dtype == np.complex128
    assert np.array_equal(out32, out64)


def test_degree_zero_untouched_and_empty():
    w = W.make_config(2, N=64, ncols=4)
    out = oracle.chase_filter(_np(w.H), _np(w.V0), np.zeros(4, np.int32), w.a, w.b, w.lambda1)
    assert np.array_equal(out, _np(w.V0))
    out = oracle.chase_filter(_np(w.H), _np(w.V0)[:, :0], np.zeros(0, np.int32), w.a, w.b, w.lambda1)
    assert out.shape == (64, 0)


def test_ragged_row_and_column_chunks():
    """N and ncols that are not multiples of the oracle's chunk sizes, vs numpy matmul recurrence."""
    N, n = 517, 37
    H = _np(W.hermitian_gaussian_ensemble(N, torch.float64, seed=51))
    V0 = _np(W.gaussian_colmajor(N, n, torch.float64, seed=52))
    a, b, l1 = -1.6, 2.1, -2.05
    m = 6
    c, e = (a + b) / 2, (b - a) / 2
    s1 = e / (l1 - c)
    A = H - c * np.eye(N)
    Vp, Vc, s = V0, (s1 / e) * (A @ V0), s1
    for _ in range(2, m + 1):
        t = 1 / (2 / s1 - s)
        Vp, Vc = Vc, (2 * t / e) * (A @ Vc) - t * s * Vp
        s = t
    out = oracle.chase_filter(H, V0, np.full(n, m, np.int32), a, b, l1)
    assert rel_fro(out, Vc) < 1e-13
