"""Alg. 5 degree optimisation (Eq. 8 :358) -- host helper chase_degrees.

Pins of the oracle: hand-computed cases where rho is an exact power of two, and the defining
property of Eq. (8) (the raw degree is the smallest m with Res / rho^m <= tol).  Then the C-ABI
function against the oracle on fuzzed inputs, incl. Table 1's degMax/degExtra."""
import math
import os

import numpy as np
import pytest

import oracle
import paper_1805_10121_b200 as pkg

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _table1():
    out = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "table1_defaults.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, d, s = line.split()
        out[k] = (float(d), float(s))
    return out


def test_oracle_hand_cases():
    # [a, b] = [-1, 1] => c = 0, e = 1, t = lambda.  t = -1.25 => rho = 1.25 + 0.75 = 2 exactly.
    a, b, lam, tol = -1.0, 1.0, -1.25, 1e-10
    mk = lambda q: tol * 2.0 ** q
    deg, order = oracle.chase_degrees([mk(10), mk(10.5), mk(3), mk(40), mk(0.25)], [lam] * 5, tol, a, b, 2, 36)
    # ceil(10)+2 = 12; ceil(10.5)+2 = 13 -> 14; ceil(3)+2 = 5 -> 6; min(42, 36) = 36; ceil(.25)+2 = 3 -> 4
    assert deg == [12, 14, 6, 36, 4]
    assert order == [4, 2, 0, 1, 3]
    # t = +1.25 (above b) has the same rho; t inside [-1, 1] has |rho| = 1 -> degMax
    assert oracle.chase_degrees([mk(10)], [1.25], tol, a, b, 2, 36)[0] == [12]
    assert oracle.chase_degrees([mk(10)], [0.3], tol, a, b, 2, 36)[0] == [36]
    # odd degMax: line 6 still rounds up to even, as printed
    assert oracle.chase_degrees([mk(40)], [lam], tol, a, b, 2, 17)[0] == [18]


def test_oracle_eq8_minimality():
    """Eq. (8): m >= log(Res/tol)/log(rho); the raw degree (before degExtra) is the smallest such m."""
    rng = np.random.default_rng(3)
    a, b, tol = -1.7, 2.05, 1e-10
    c, e = (a + b) / 2, (b - a) / 2
    for _ in range(200):
        lam = rng.uniform(-2.6, a - 1e-3)
        res = 10.0 ** rng.uniform(-9.5, -1)
        d = oracle.chase_degrees([res], [lam], tol, a, b, 0, 10 ** 6)[0][0]
        t = (lam - c) / e
        rho = abs(t) + math.sqrt(t * t - 1)
        m = d - 1 if (res / rho ** (d - 1) <= tol * (1 + 1e-12) and d - 1 >= 1) else d     # undo the even rounding
        assert res / rho ** m <= tol * (1 + 1e-9)
        assert res / rho ** (m - 1) > tol * (1 - 1e-9)


def test_library_matches_oracle_fuzz():
    t1 = _table1()
    rng = np.random.default_rng(11)
    for prec in (0, 1):
        tol, deg_extra, deg_max = t1["tol"][prec], int(t1["degExtra"][prec]), int(t1["degMax"][prec])
        a, b = -1.7, 2.05
        n = 500
        ritz = rng.uniform(-2.5, 2.2, n)              # some inside [a, b], some above b
        resid = 10.0 ** rng.uniform(math.log10(tol) - 2, 0, n)     # some already below tol
        deg, perm = pkg.chase_degrees(resid, ritz, tol, a, b, deg_extra, deg_max)
        odeg, oorder = oracle.chase_degrees(resid, ritz, tol, a, b, deg_extra, deg_max)
        assert list(perm) == oorder
        assert list(deg) == [odeg[j] for j in oorder]
        assert np.all(np.diff(deg) >= 0) and np.all(deg % 2 == 0) and deg.max() <= deg_max + deg_max % 2
        assert deg.min() >= 2
        # the output is directly consumable by the filter's schedule
        m_max, off = pkg.chase_filter_schedule(deg)
        assert m_max == deg.max()


def test_library_hand_cases_and_errors():
    tol = 1e-10
    deg, perm = pkg.chase_degrees([tol * 2 ** 10, tol * 2 ** 3], [-1.25, -1.25], tol, -1.0, 1.0, 2, 36)
    assert list(deg) == [6, 12] and list(perm) == [1, 0]
    deg, perm = pkg.chase_degrees([], [], tol, -1.0, 1.0)
    assert deg.size == 0
    for kw, code in ((dict(tol=0.0), -1), (dict(a=1.0, b=1.0), -2), (dict(deg_max=0), -1), (dict(deg_extra=-1), -1)):
        args = dict(resid=[1e-3], ritzv=[-1.5], tol=tol, a=-1.0, b=1.0, deg_extra=2, deg_max=36)
        args.update(kw)
        with pytest.raises(pkg.ChaseFilterError) as ei:
            pkg.chase_degrees(**args)
        assert ei.value.code == code
    with pytest.raises(pkg.ChaseFilterError):
        pkg.chase_degrees([-1.0], [-1.5], tol, -1.0, 1.0)
