"""Maxwell equal-area construction on the oracle's equations of state.

ORACLE — TEST INFRASTRUCTURE ONLY (see oracle/lbm_oracle.cpp header).

The paper compares simulated coexistence densities with "the values obtained
from Maxwell's construction" and prints them at T_r = 0.8 for five EOS
(Table 1, last column).  This module is that definition written out:
find p_sat, rho_v < rho_l with

    p(rho_v) = p(rho_l) = p_sat   and   int_{v_l}^{v_v} (p(1/v) - p_sat) dv = 0,

with p(rho) evaluated by the C++ oracle's ``olbm_eos_pressure`` (so the printed
Table 1 values pin the C++ EOS formulas and parameters).
"""
from __future__ import annotations

import numpy as np
from scipy.optimize import brentq

from . import lbm_oracle as _o

_GL_X, _GL_W = np.polynomial.legendre.leggauss(24)


def _rho_max(kind: str, b: float) -> float:
    # cubic EOS diverge at b*rho = 1; Carnahan-Starling at eta = b*rho/4 = 1
    return (4.0 / b if kind == "CS" else 1.0 / b) * (1.0 - 1e-9)


def spinodals(kind, a, b, R, omega, T, n=400001):
    """Vapour-side local maximum and liquid-side local minimum of p(rho)."""
    rmax = _rho_max(kind, b)
    rho = np.linspace(rmax * 1e-7, rmax * 0.98, n)
    p = _o.eos_pressure(kind, a, b, R, omega, T, rho)
    dp = np.diff(p)
    imax = np.where((dp[:-1] > 0) & (dp[1:] <= 0))[0]
    imin = np.where((dp[:-1] < 0) & (dp[1:] >= 0))[0]
    if len(imax) == 0 or len(imin) == 0:
        raise ValueError("no van der Waals loop: T is above the critical temperature")
    i1 = imax[0] + 1
    i2 = imin[imin > i1][0] + 1
    return rho[i1], rho[i2], p[i1], p[i2]


def _area(p_fn, p_sat, rho_v, rho_l, panels=200):
    # int_{v_l}^{v_v} (p(1/v) - p_sat) dv on log-spaced panels, Gauss-Legendre per panel
    edges = np.exp(np.linspace(np.log(1.0 / rho_l), np.log(1.0 / rho_v), panels + 1))
    lo, hi = edges[:-1, None], edges[1:, None]
    v = 0.5 * (hi + lo) + 0.5 * (hi - lo) * _GL_X[None, :]
    wts = 0.5 * (hi - lo) * _GL_W[None, :]
    return float(np.sum(wts * (p_fn(1.0 / v.reshape(-1)).reshape(v.shape) - p_sat)))


def coexistence(kind: str, a: float, b: float, R: float, omega: float, T: float):
    """Return (rho_v, rho_l, p_sat) of the Maxwell construction."""
    def p_fn(r):
        return _o.eos_pressure(kind, a, b, R, omega, T, r)

    def p1(r):
        return float(p_fn(np.array([r]))[0])

    rs1, rs2, pmax, pmin = spinodals(kind, a, b, R, omega, T)
    rmax = _rho_max(kind, b)
    p_lo = max(pmin, 0.0) + 1e-14 * pmax
    p_hi = pmax * (1.0 - 1e-12)

    def branches(ps):
        rv = brentq(lambda r: p1(r) - ps, 1e-300, rs1, xtol=1e-300, rtol=1e-14)
        rl = brentq(lambda r: p1(r) - ps, rs2, rmax * 0.999999, xtol=1e-16, rtol=1e-14)
        return rv, rl

    def g(ps):
        rv, rl = branches(ps)
        return _area(p_fn, ps, rv, rl)

    ps = brentq(g, p_lo, p_hi, xtol=1e-18, rtol=1e-13)
    rv, rl = branches(ps)
    return rv, rl, ps
