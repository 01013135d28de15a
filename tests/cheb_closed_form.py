"""Closed forms from the paper, retyped independently of oracle/ and of the CUDA path.

Used only by tests to pin the oracle (and, at full size, the GPU result).
  C_m(t) = cosh(m acosh t) for |t| > 1 (with sign(t)^m), cos(m acos t) on [-1, 1]
      -- Def. 4.1, Eq. (2)
  p_m(x) = C_m((x - c)/e) / C_m((gamma - c)/e)     -- Eq. (5)
  gamma = mu_1 = lambda1, alpha = mu_{nev+nex} = a, beta = b_sup = b   -- PAPER.md:305
"""
import numpy as np


def cheb_C(m: int, t):
    t = np.asarray(t, dtype=np.float64)
    out = np.empty_like(t)
    inside = np.abs(t) <= 1.0
    out[inside] = np.cos(m * np.arccos(t[inside]))
    to = t[~inside]
    out[~inside] = np.sign(to) ** m * np.cosh(m * np.arccosh(np.abs(to)))
    return out


def p_m(m: int, x, a: float, b: float, lambda1: float):
    c = (a + b) / 2.0
    e = (b - a) / 2.0
    return cheb_C(m, (np.asarray(x, dtype=np.float64) - c) / e) / cheb_C(m, np.array([(lambda1 - c) / e]))[0]


def rel_fro(x, ref) -> float:
    return float(np.linalg.norm(np.asarray(x) - np.asarray(ref)) / np.linalg.norm(np.asarray(ref)))
