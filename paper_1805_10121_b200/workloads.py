"""Seeded synthetic inputs for the Chebyshev-filter hot path (ChASE, arXiv 1805.10121).

This module is the ONLY code shared by the CUDA path and the CPU oracle.  It holds
input generation and nothing of the method's arithmetic: no Chebyshev scalars, no
recurrence, no matrix-vector product of the filter.  Recipes follow DESIGN.md
("Input recipe") and BASELINE.json `configs`; they stand in for the paper's DFT
(NaCl, AuAg) and BSE matrices, which are not available.

Layout convention: every matrix is COLUMN-MAJOR with leading dimension N (Listing 2,
PAPER.md:563-566).  A torch tensor returned here has shape (rows, cols) and strides
(1, rows), i.e. it is the transpose-view of a contiguous (cols, rows) tensor, so
`t.data_ptr()` addresses element (i, j) at offset i + j*rows and `t.numpy()` is
Fortran-contiguous without a copy.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import torch

BASE_SEED = 180510121  # seed = BASE_SEED + 1000*cfg (+0 H, +1 V0, +2 degrees)

_REAL_OF = {
    torch.complex128: torch.float64,
    torch.complex64: torch.float32,
    torch.float64: torch.float64,
    torch.float32: torch.float32,
}
DTYPE_NAMES = {
    torch.float32: "f32",
    torch.float64: "f64",
    torch.complex64: "c64",
    torch.complex128: "c128",
}


@dataclasses.dataclass
class Workload:
    """One filter call's inputs.  H, V0 are column-major torch tensors (see module doc)."""

    name: str
    H: torch.Tensor            # N x N, Hermitian, full storage
    V0: torch.Tensor           # N x ncols
    degrees: torch.Tensor      # int32 [ncols], host, non-decreasing
    a: float                   # mu_{nev+nex}: lower edge of the damped interval
    b: float                   # b_sup: upper bound of the spectrum
    lambda1: float             # mu_1: lower end of the wanted spectrum
    dtype: torch.dtype
    eigvals: Optional[torch.Tensor] = None   # known spectrum (real, ascending) if constructed
    eigvecs: Optional[torch.Tensor] = None   # known eigenvectors (columns), if constructed

    @property
    def N(self) -> int:
        return self.H.shape[0]

    @property
    def ncols(self) -> int:
        return self.V0.shape[1]

    @property
    def sum_deg(self) -> int:
        return int(self.degrees.sum().item())

    def flops(self) -> float:
        """Metric flops (BASELINE.json): f*N^2*sum(deg), f = 8 complex / 2 real."""
        f = 8.0 if self.dtype.is_complex else 2.0
        return f * float(self.N) ** 2 * float(self.sum_deg)


def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return g


def empty_colmajor(rows: int, cols: int, dtype, device="cpu") -> torch.Tensor:
    """rows x cols tensor with strides (1, rows) (column-major, ld = rows)."""
    return torch.empty((cols, rows), dtype=dtype, device=device).t()


def as_colmajor(x: torch.Tensor) -> torch.Tensor:
    """Copy a 2-D tensor into column-major storage."""
    out = empty_colmajor(x.shape[0], x.shape[1], x.dtype, x.device)
    out.copy_(x)
    return out


def is_colmajor(x: torch.Tensor) -> bool:
    return x.dim() == 2 and x.stride(0) == 1 and (x.shape[1] <= 1 or x.stride(1) == x.shape[0])


def gaussian_colmajor(rows: int, cols: int, dtype, seed: int, device="cpu",
                      std: float = 1.0, panel: int = 4096) -> torch.Tensor:
    """i.i.d. Gaussian entries, E|x|^2 = std^2 (complex: re and im each std^2/2),
    generated panel-by-panel (in FP64, then rounded to `dtype`) so that big matrices
    never need a second full-size temporary."""
    g = _gen(seed, device)
    out = empty_colmajor(rows, cols, dtype, device)
    store = out.t()  # contiguous (cols, rows)
    gen_dtype = torch.complex128 if dtype.is_complex else torch.float64
    for j0 in range(0, cols, panel):
        j1 = min(cols, j0 + panel)
        blk = torch.randn((j1 - j0, rows), dtype=gen_dtype, device=device, generator=g)
        store[j0:j1].copy_(blk * std)
    return out


def hermitian_gaussian_ensemble(N: int, dtype, seed: int, device="cpu",
                                block: int = 4096) -> torch.Tensor:
    """GUE (complex dtype) / GOE (real dtype) with off-diagonal E|H_ij|^2 = 1/N
    (reading G14): G_ij i.i.d. with E|G_ij|^2 = 1/N, H = (G + G^H)/sqrt(2),
    diagonal forced real.  Spectrum ~ semicircle on [-2, 2].  Symmetrised in place
    block by block; the result is bitwise Hermitian (H[i,j] == conj(H[j,i]))."""
    H = gaussian_colmajor(N, N, dtype, seed, device, std=1.0 / math.sqrt(N), panel=block)
    r = 1.0 / math.sqrt(2.0)
    for i0 in range(0, N, block):
        i1 = min(N, i0 + block)
        for j0 in range(i0, N, block):
            j1 = min(N, j0 + block)
            upper = H[i0:i1, j0:j1]
            lower = H[j0:j1, i0:i1]
            if i0 == j0:
                s = (upper + upper.mH) * r
                # make the diagonal block bitwise Hermitian: take the upper triangle
                s = torch.triu(s) + torch.triu(s, 1).mH
                if dtype.is_complex:
                    d = torch.arange(i1 - i0, device=s.device)
                    s[d, d] = s[d, d].real.to(s.dtype)
                upper.copy_(s)
            else:
                s = (upper + lower.mH) * r
                upper.copy_(s)
                lower.copy_(s.mH)
    return H


def known_spectrum_hermitian(N: int, dtype, seed: int, device="cpu"):
    """cfg-1 construction: H = Q diag(lam) Q^H, lam ~ sorted i.i.d. U(-1,1), Q from the
    QR factorisation of a seeded Gaussian matrix; then (H + H^H)/2 with a real diagonal.
    Returns (H column-major, lam ascending [real], Q)."""
    g = _gen(seed, device)
    rdt = _REAL_OF[dtype]
    lam = (torch.rand(N, dtype=torch.float64, device=device, generator=g) * 2.0 - 1.0)
    lam, _ = torch.sort(lam)
    wide = torch.complex128 if dtype.is_complex else torch.float64
    G = torch.randn((N, N), dtype=wide, device=device, generator=g)
    Q, _ = torch.linalg.qr(G)
    Hd = (Q * lam.to(wide)) @ Q.mH
    Hd = (Hd + Hd.mH) * 0.5
    Hd = torch.triu(Hd) + torch.triu(Hd, 1).mH
    if dtype.is_complex:
        d = torch.arange(N, device=device)
        Hd[d, d] = Hd[d, d].real.to(wide)
    H = as_colmajor(Hd.to(dtype))
    return H, lam.to(rdt), Q


def sorted_even_degrees(ncols: int, lo: int, hi: int, seed: int) -> torch.Tensor:
    """Even degrees drawn i.i.d. uniformly from {lo, lo+2, ..., hi}, sorted ascending
    (Alg. 1 line 15; even-ness: Alg. 5 line 6)."""
    g = _gen(seed, "cpu")
    nvals = (hi - lo) // 2 + 1
    idx = torch.randint(0, nvals, (ncols,), generator=g)
    deg, _ = torch.sort(lo + 2 * idx)
    return deg.to(torch.int32)


def uniform_degrees(ncols: int, m: int) -> torch.Tensor:
    return torch.full((ncols,), m, dtype=torch.int32)


# --------------------------------------------------------------------------------------
# The five BASELINE.json configs.  `N`/`ncols` may be overridden to get a reduced-size
# case with the same recipe (used by tests so the oracle finishes in seconds).
# --------------------------------------------------------------------------------------

CONFIG_SHAPES = {
    1: dict(N=512, ncols=60, dtype=torch.complex128),
    2: dict(N=4096, ncols=256, dtype=torch.complex128),
    3: dict(N=20000, ncols=1400, dtype=torch.float64),
    4: dict(N=40000, ncols=2000, dtype=torch.complex128),
    5: dict(N=60000, ncols=3000, dtype=torch.complex64),
}


def make_config(cfg: int, device="cpu", N: Optional[int] = None, ncols: Optional[int] = None,
                dtype: Optional[torch.dtype] = None) -> Workload:
    shape = CONFIG_SHAPES[cfg]
    N = shape["N"] if N is None else N
    ncols = shape["ncols"] if ncols is None else ncols
    dtype = shape["dtype"] if dtype is None else dtype
    seed = BASE_SEED + 1000 * cfg
    name = f"cfg{cfg}:N={N},ncols={ncols},{DTYPE_NAMES[dtype]}"

    if cfg == 1:
        # H = Q diag(lam) Q^H, lam sorted U(-1,1); a = lam_{ncols+1}, b = lam_N, lambda1 = lam_1
        # (1-based; reading G13).  Uniform degree 10.
        H, lam, Q = known_spectrum_hermitian(N, dtype, seed, device)
        V0 = gaussian_colmajor(N, ncols, dtype, seed + 1, device)
        return Workload(name, H, V0, uniform_degrees(ncols, 10),
                        a=float(lam[ncols]), b=float(lam[N - 1]), lambda1=float(lam[0]),
                        dtype=dtype, eigvals=lam, eigvecs=Q)
    if cfg == 2:
        H = hermitian_gaussian_ensemble(N, dtype, seed, device)
        V0 = gaussian_colmajor(N, ncols, dtype, seed + 1, device)
        return Workload(name, H, V0, sorted_even_degrees(ncols, 10, 30, seed + 2),
                        a=-1.6, b=2.05, lambda1=-2.0, dtype=dtype)
    if cfg == 3:
        # GOE + the N/20 smallest diagonal entries overwritten with -3 (reading G15).
        H = hermitian_gaussian_ensemble(N, dtype, seed, device)
        diag = torch.diagonal(H).real.clone() if dtype.is_complex else torch.diagonal(H).clone()
        order = torch.sort(diag, stable=True).indices[: N // 20]
        H[order, order] = torch.full((order.numel(),), -3.0, dtype=dtype, device=H.device)
        V0 = gaussian_colmajor(N, ncols, dtype, seed + 1, device)
        return Workload(name, H, V0, uniform_degrees(ncols, 20),
                        a=-2.0, b=2.05, lambda1=-3.1, dtype=dtype)
    if cfg == 4:
        H = hermitian_gaussian_ensemble(N, dtype, seed, device)
        V0 = gaussian_colmajor(N, ncols, dtype, seed + 1, device)
        return Workload(name, H, V0, sorted_even_degrees(ncols, 8, 36, seed + 2),
                        a=-1.7, b=2.05, lambda1=-2.0, dtype=dtype)
    if cfg == 5:
        H = hermitian_gaussian_ensemble(N, dtype, seed, device)
        V0 = gaussian_colmajor(N, ncols, dtype, seed + 1, device)
        return Workload(name, H, V0, uniform_degrees(ncols, 16),
                        a=-1.75, b=2.05, lambda1=-2.0, dtype=dtype)
    raise ValueError(f"unknown config {cfg}")


def reflector_hermitian(N: int, dtype, seed: int, device="cpu", nreflect: int = 2):
    """Dense Hermitian H = R diag(lam) R^H with R a product of `nreflect` Householder
    reflectors I - 2 u u^H (|u| = 1): exactly known eigenpairs, built in O(N^2) without
    a factorisation (pin P6 at sizes where QR/eigh are too slow).
    Returns (H column-major, lam [float64, ascending], list of unit vectors u)."""
    g = _gen(seed, device)
    wide = torch.complex128 if dtype.is_complex else torch.float64
    lam, _ = torch.sort(torch.rand(N, dtype=torch.float64, device=device, generator=g) * 4.0 - 2.0)
    us = []
    for _ in range(nreflect):
        u = torch.randn(N, dtype=wide, device=device, generator=g)
        us.append(u / torch.linalg.vector_norm(u))
    # H = R D R^H with R = R_1 R_2 ...: apply the reflectors to diag(lam) from both sides.
    Hd = torch.diag(lam.to(wide))
    for u in reversed(us):
        Hd = Hd - 2.0 * torch.outer(u, u.conj() @ Hd)       # R_i * Hd
        Hd = Hd - 2.0 * torch.outer(Hd @ u, u.conj())       # Hd * R_i^H (R_i Hermitian)
    Hd = (Hd + Hd.mH) * 0.5
    Hd = torch.triu(Hd) + torch.triu(Hd, 1).mH
    if dtype.is_complex:
        d = torch.arange(N, device=device)
        Hd[d, d] = Hd[d, d].real.to(wide)
    return as_colmajor(Hd.to(dtype)), lam, us


def parity_sample_columns(degrees, min_cols: int = 32, tile_widths=(64, 128), seed: int = BASE_SEED + 7):
    """Column sample for parity at sizes where the oracle cannot run the full block (SURVEY 8(c)
    "Where the oracle runs in full vs sampled"): the first and last column of EVERY distinct degree
    (i.e. both sides of every column drop of Alg. 4 l.12-14), the global first / last column, the
    columns at -1 / 0 / +1 around the first multiples of the kernels' column-tile widths, the middle
    column, and seeded random columns up to `min_cols`.  Returns sorted unique indices; each sampled
    column keeps its own degree (columns are independent, pin P7)."""
    deg = [int(d) for d in (degrees.tolist() if hasattr(degrees, "tolist") else degrees)]
    n = len(deg)
    if n == 0:
        return []
    cols = {0, n - 1, n // 2}
    for j in range(n):
        if j == 0 or deg[j] != deg[j - 1]:
            cols.add(j)
            if j > 0:
                cols.add(j - 1)
    for w in tile_widths:
        for mult in (1, 2):
            for d in (-1, 0, 1):
                cols.add(w * mult + d)
    cols = {c for c in cols if 0 <= c < n}
    g = _gen(seed, "cpu")
    while len(cols) < min(min_cols, n):
        cols.add(int(torch.randint(0, n, (1,), generator=g).item()))
    return sorted(cols)
