"""ORACLE -- TEST INFRASTRUCTURE ONLY (see chase_filter_oracle.c for the full header).

ctypes front end to the plain-C FP64 oracle of the ChASE Chebyshev filter
(Alg. 4, Eq. (7)).  It imports nothing from the
product package and the product package imports nothing from here.  Allowed callers:
tests/, __graft_entry__.smoke(), bench.py's cpu_baseline / --impl reference legs.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "chase_filter_oracle.c")
_LIB = os.path.join(_DIR, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp; no -march so the same .so runs on any x86-64 host."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-Wall",
                               "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_chase_scalars.restype = None
        lib.oracle_chase_scalars.argtypes = [ctypes.c_double] * 3 + [ctypes.c_int] + [ctypes.c_void_p] * 5
        lib.oracle_chase_filter.restype = ctypes.c_int
        lib.oracle_chase_filter.argtypes = [
            ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int64,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p,
            ctypes.c_double, ctypes.c_double, ctypes.c_double]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def chase_scalars(a: float, b: float, lambda1: float, m_max: int):
    """(sigma[1..m], alpha[1..m], beta[1..m], c, e) of Alg. 4; arrays have length m_max+1, entry 0 unused."""
    lib = _load()
    sigma = np.zeros(m_max + 1)
    alpha = np.zeros(m_max + 1)
    beta = np.zeros(m_max + 1)
    c = ctypes.c_double()
    e = ctypes.c_double()
    lib.oracle_chase_scalars(a, b, lambda1, m_max, sigma.ctypes.data, alpha.ctypes.data,
                             beta.ctypes.data, ctypes.addressof(c), ctypes.addressof(e))
    return sigma, alpha, beta, c.value, e.value


def chase_filter(H: np.ndarray, V0: np.ndarray, degrees, a: float, b: float, lambda1: float) -> np.ndarray:
    """out[:, j] = p_{degrees[j]}(H) V0[:, j], FP64, returned as a new Fortran-ordered array.

    H: N x N, Fortran-contiguous, dtype float64/complex128 (used as is) or
       float32/complex64 (upcast element-wise inside the C loop).
    V0: N x ncols, any float/complex dtype; upcast to FP64 (complex iff H is complex).
    """
    lib = _load()
    H = np.asarray(H)
    if H.ndim != 2 or H.shape[0] != H.shape[1]:
        raise ValueError("H must be square")
    if not H.flags.f_contiguous:
        H = np.asfortranarray(H)
    is_complex = np.iscomplexobj(H)
    h_is_f32 = H.dtype in (np.float32, np.complex64)
    if H.dtype not in (np.float32, np.float64, np.complex64, np.complex128):
        raise ValueError(f"unsupported H dtype {H.dtype}")
    N = H.shape[0]
    wide = np.complex128 if is_complex else np.float64
    if np.iscomplexobj(V0) and not is_complex:
        raise ValueError("complex V0 with real H")
    V = np.array(V0, dtype=wide, order="F", copy=True)
    if V.ndim != 2 or V.shape[0] != N:
        raise ValueError("V0 must be N x ncols")
    W = np.empty_like(V, order="F")
    deg = np.ascontiguousarray(np.asarray(degrees, dtype=np.int32))
    if deg.shape != (V.shape[1],):
        raise ValueError("degrees must have one entry per column")
    rc = lib.oracle_chase_filter(H.ctypes.data, int(h_is_f32), int(is_complex), N,
                                 V.ctypes.data, W.ctypes.data, V.shape[1], deg.ctypes.data,
                                 float(a), float(b), float(lambda1))
    if rc != 0:
        raise RuntimeError(f"oracle_chase_filter failed: {rc}")
    return V


def chase_degrees(resid, ritzv, tol: float, a: float, b: float, deg_extra: int = 2, deg_max: int = 36):
    """ORACLE for Alg. 5 "Degree Optimization" (Eq. (8)) and the
    sort by degree of Alg. 1 l.15, written line by line in the paper's notation.
    Returns (deg unsorted [list of int], order [stable argsort by degree]).

    Reading (G17): for |t| <= 1 the two roots t +- sqrt(t^2-1) are complex of modulus 1,
    so |rho| = 1, log|rho| = 0 and line 4 is unbounded: line 5's cap gives deg = DEGMAX.
    """
    import cmath
    import math
    c = (a + b) / 2.0
    e = (b - a) / 2.0
    deg = []
    for res, lam in zip(resid, ritzv):
        t = (lam - c) / e                                                    # l.2
        root = cmath.sqrt(t * t - 1.0)
        rho = max(abs(t - root), abs(t + root))                              # l.3
        if rho <= 1.0 + 1e-300 or math.log(rho) == 0.0:
            d = float("inf")
        else:
            d = math.ceil(abs(math.log(res / tol) / math.log(rho)))          # l.4
        d = min(d + deg_extra, deg_max)                                      # l.5
        d = int(d)
        deg.append(d + d % 2)                                                # l.6
    order = sorted(range(len(deg)), key=lambda j: deg[j])                    # Alg. 1 l.15 (stable)
    return deg, order


def hemm(H: np.ndarray, X: np.ndarray, Y, alpha: float = 1.0, beta: float = 0.0, shift=0.0) -> np.ndarray:
    """ORACLE: alpha (H X - X diag(shift)) + beta Y in FP64 (Listing 1 HEMM), new array.
    `shift` is a scalar or one value per column."""
    lib = _load()
    lib.oracle_hemm.restype = ctypes.c_int
    lib.oracle_hemm.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int64, ctypes.c_void_p,
                                ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_void_p]
    H = np.asarray(H)
    if not H.flags.f_contiguous:
        H = np.asfortranarray(H)
    is_complex = np.iscomplexobj(H)
    h_is_f32 = H.dtype in (np.float32, np.complex64)
    wide = np.complex128 if is_complex else np.float64
    Xw = np.array(X, dtype=wide, order="F", copy=True)
    N, n = Xw.shape
    Yw = np.zeros((N, n), dtype=wide, order="F") if Y is None else np.array(Y, dtype=wide, order="F", copy=True)
    sh = np.ascontiguousarray(np.broadcast_to(np.asarray(shift, dtype=np.float64), (n,)))
    rc = lib.oracle_hemm(H.ctypes.data, int(h_is_f32), int(is_complex), N, Xw.ctypes.data, Yw.ctypes.data, n,
                         float(alpha), float(beta), sh.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"oracle_hemm failed: {rc}")
    return Yw


def residuals(H: np.ndarray, V: np.ndarray, ritzv) -> np.ndarray:
    """ORACLE: resid[j] = ||H v_j - ritzv[j] v_j||_2 (Alg. 1 l.8; Resd)."""
    R = hemm(H, V, None, 1.0, 0.0, np.asarray(ritzv, dtype=np.float64))
    return np.sqrt(np.sum(R.real ** 2 + R.imag ** 2, axis=0))
