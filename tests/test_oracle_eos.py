"""Pins for the oracle's equations of state and the Maxwell construction (CPU only)."""
from pathlib import Path

import numpy as np
import pytest

from oracle import lbm_oracle as o
from oracle import maxwell as mx
from paper_2506_17713_b200 import workloads as W

GOLD = Path(__file__).parent / "golden"

# Yuan & Schaefer parameters as quoted by the paper
PARAMS = {
    "CS": dict(a=1.0, b=4.0, R=1.0, omega=0.0),
    "PR": dict(a=2 / 49, b=2 / 21, R=1.0, omega=0.344),
    "RK": dict(a=2 / 49, b=2 / 21, R=1.0, omega=0.0),
    "RKS": dict(a=2 / 49, b=2 / 21, R=1.0, omega=0.344),
    "VDW": dict(a=9 / 49, b=2 / 21, R=1.0, omega=0.0),
}


def _table1():
    rows = {}
    for line in (GOLD / "table1_maxwell.txt").read_text().splitlines():
        if line and not line.startswith("#"):
            k, g, l = line.split()
            rows[k] = (float(g), float(l))
    return rows


@pytest.mark.parametrize("kind", ["CS", "PR", "RK", "RKS", "VDW"])
def test_maxwell_densities_match_paper_table1(kind):
    """Paper Table 1, last column, T_r = 0.8.  The table prints 4 decimals;
    agreement is to +-1.5 units of the last printed digit."""
    p = PARAMS[kind]
    Tc = o.eos_critical_temperature(kind, p["a"], p["b"], p["R"])
    rv, rl, ps = mx.coexistence(kind, p["a"], p["b"], p["R"], p["omega"], 0.8 * Tc)
    g, l = _table1()[kind]
    assert abs(rv - g) <= 1.5e-4
    assert abs(rl - l) <= 1.5e-4
    # the construction itself: equal pressures on both branches
    pv, pl = o.eos_pressure(kind, p["a"], p["b"], p["R"], p["omega"], 0.8 * Tc, [rv, rl])
    assert abs(pv - ps) < 1e-12 and abs(pl - ps) < 1e-12


@pytest.mark.parametrize("kind", ["CS", "PR", "RK", "RKS", "VDW"])
def test_critical_point_is_an_inflection(kind):
    """At T = T_c the isotherm has dp/drho = d2p/drho2 = 0 at the critical density (textbook definition);
    pins the T_c formulas independently of Table 1.  CS/PR constants are rounded (0.3773, 0.0778/0.45724),
    hence the tolerance."""
    p = PARAMS[kind]
    Tc = o.eos_critical_temperature(kind, p["a"], p["b"], p["R"])
    rmax = (4.0 if kind == "CS" else 1.0) / p["b"]
    rho = np.linspace(0.02 * rmax, 0.6 * rmax, 20001)
    pr = o.eos_pressure(kind, p["a"], p["b"], p["R"], p["omega"], Tc, rho)
    dp = np.gradient(pr, rho)
    i = np.argmin(dp)
    # minimum slope is ~0 relative to the ideal-gas slope R*T_c
    assert abs(dp[i]) < 2e-3 * p["R"] * Tc
    # slightly above T_c the isotherm is monotone, slightly below it has a loop
    pa = o.eos_pressure(kind, p["a"], p["b"], p["R"], p["omega"], 1.01 * Tc, rho)
    pb = o.eos_pressure(kind, p["a"], p["b"], p["R"], p["omega"], 0.99 * Tc, rho)
    assert np.all(np.diff(pa) > 0)
    assert np.any(np.diff(pb) < 0)


def test_vdw_critical_constants_closed_form():
    a, b, R = 9 / 49, 2 / 21, 1.0
    Tc = o.eos_critical_temperature("VDW", a, b, R)
    assert abs(Tc - 8 * a / (27 * b * R)) < 1e-15
    pc = o.eos_pressure("VDW", a, b, R, 0.0, Tc, [1 / (3 * b)])[0]
    assert abs(pc - a / (27 * b * b)) < 1e-13


@pytest.mark.parametrize("kind", ["CS", "PR", "RK", "RKS", "VDW"])
def test_ideal_gas_limit(kind):
    p = PARAMS[kind]
    T = 0.07
    rho = np.array([1e-7, 1e-6])
    pr = o.eos_pressure(kind, p["a"], p["b"], p["R"], p["omega"], T, rho)
    assert np.allclose(pr / (rho * p["R"] * T), 1.0, atol=1e-5)


def test_workload_constants_match_maxwell():
    Tc = o.eos_critical_temperature("CS", W.CS_A, W.CS_B, W.CS_R)
    assert abs(W.CS_T_085 - 0.85 * Tc) < 1e-9
    rv, rl, _ = mx.coexistence("CS", W.CS_A, W.CS_B, W.CS_R, 0.0, W.CS_T_085)
    assert abs(rv - W.CS_RHO_V_085) < 1e-6 and abs(rl - W.CS_RHO_L_085) < 1e-6
    Tc = o.eos_critical_temperature("PR", W.PR_A, W.PR_B, W.PR_R)
    assert abs(W.PR_T_07 - 0.7 * Tc) < 1e-9
    rv, rl, _ = mx.coexistence("PR", W.PR_A, W.PR_B, W.PR_R, W.PR_OMEGA, W.PR_T_07)
    assert abs(rv - W.PR_RHO_V_07) < 1e-6 and abs(rl - W.PR_RHO_L_07) < 1e-6


@pytest.mark.parametrize("kind,alpha", [("CS", 1.0), ("PR", 0.5)])
def test_pseudopotential_reproduces_eos_pressure(kind, alpha):
    """Eq. 12: with psi = sqrt(2(alpha p_EOS - c_s^2 rho)/g_kk) the model pressure
    c_s^2 rho + (g_kk/2) psi^2 is alpha * p_EOS wherever the radicand is positive (g_kk = -1)."""
    p = PARAMS[kind]
    Tc = o.eos_critical_temperature(kind, p["a"], p["b"], p["R"])
    T = 0.85 * Tc
    n = 64
    rmax = (4.0 if kind == "CS" else 1.0) / p["b"]
    rho = np.linspace(0.01 * rmax, 0.5 * rmax, n)
    wl = dict(lattice="D2Q9", nx=n, ny=1, nz=1, n_components=1, periodic=(True, True, True), psi_kind=[kind],
              eos=[dict(a=p["a"], b=p["b"], R=p["R"], omega=p["omega"], T=T, alpha=alpha)], G=[[-1.0]],
              collision="BGK", tau=[1.0], forcing="EDM", compute_dtype="f64", store_dtype="f64")
    s = o.Oracle(wl)
    s.init_fields([rho])
    _, _, pm = s.get_macroscopic()
    pe = alpha * o.eos_pressure(kind, p["a"], p["b"], p["R"], p["omega"], T, rho)
    psi = s.get_psi(0)
    ok = psi > 0
    assert ok.sum() > n // 2
    assert np.allclose(pm[ok], pe[ok], rtol=0, atol=1e-14)
    # where alpha p - c_s^2 rho >= 0 the root is clamped (reading R4) and p falls back to c_s^2 rho
    assert np.allclose(pm[~ok], rho[~ok] / 3.0, rtol=0, atol=1e-15)


def test_psi_kinds_closed_form():
    rho = np.array([0.05, 0.5, 1.0, 3.0])
    def run(kind, **eos):
        wl = dict(lattice="D2Q9", nx=4, ny=1, nz=1, n_components=1, periodic=(True, True, True), psi_kind=[kind],
                  eos=[eos], G=[[-1.0]], collision="BGK", tau=[1.0], forcing="EDM", compute_dtype="f64",
                  store_dtype="f64")
        s = o.Oracle(wl)
        s.init_fields([rho])
        return s.get_psi(0)
    assert np.allclose(run("RHO"), rho, rtol=0, atol=1e-15)
    assert np.allclose(run("EXP"), np.exp(-1 / rho), rtol=0, atol=1e-15)
    assert np.allclose(run("SC93", rho0=2.0), 2.0 * (1 - np.exp(-rho / 2.0)), rtol=0, atol=1e-15)
