"""Physics pins: the oracle's whole step against what the paper and the mathematics fix (CPU only).

Runs are sized to finish in about a minute in total.
"""
from pathlib import Path

import numpy as np
import pytest
from scipy.optimize import brentq

from conftest import make_oracle
from oracle import lbm_oracle as o
from paper_2506_17713_b200 import workloads as W
from test_oracle_basics import base_wl

GOLD = Path(__file__).parent / "golden"


def _scalars():
    out = {}
    for line in (GOLD / "paper_scalars.txt").read_text().splitlines():
        if line and not line.startswith("#"):
            parts = line.split()
            out[parts[0]] = (float(parts[1]), float(parts[2]))
    return out


def _flat(nx, ny, rho_l, rho_v, w=3.0):
    x = np.tile(np.arange(nx), ny).astype(float)
    return W.tanh_profile(np.abs(x - (nx - 1) / 2), nx / 4, w, rho_l, rho_v)


def test_flat_interface_cs_coexistence_vs_maxwell():
    """CS at T_r = 0.85, plain Shan-Chen force (A = 0): liquid within 0.5 % of Maxwell, vapour low by
    several % (the A-weighted Zhang-Chen term that the paper tunes, is NEXT-1).  Also: the bulk
    pressures of both phases agree (mechanical equilibrium) -- this pins the force normalisation R2,
    because p = c_s^2 rho + (g/2) psi^2 only holds if sum_i G_i e_i e_i = I."""
    nx, ny = 128, 2
    wl = base_wl("D2Q9", (nx, ny, 1), psi_kind=["CS"], eos=[dict(a=W.CS_A, b=W.CS_B, R=W.CS_R, T=W.CS_T_085)],
                 G=[[-1.0]])
    s = make_oracle(wl, dict(rho=[_flat(nx, ny, W.CS_RHO_L_085, W.CS_RHO_V_085)]))
    s.step(8000)
    rho, u, p = s.get_macroscopic()
    r, pp = rho[0].reshape(ny, nx)[0], p.reshape(ny, nx)[0]
    assert abs(r[nx // 2] / W.CS_RHO_L_085 - 1) < 5e-3
    assert -0.12 < r[0] / W.CS_RHO_V_085 - 1 < 0.0
    assert abs(pp[nx // 2] - pp[0]) < 2e-3 * pp[0]
    assert np.abs(u).max() < _scalars()["spurious_current_max"][0]


def test_edm_coexistence_independent_of_tau():
    nx, ny = 96, 2
    out = []
    for tau in (1.0, 0.8):
        wl = base_wl("D2Q9", (nx, ny, 1), psi_kind=["CS"], eos=[dict(a=W.CS_A, b=W.CS_B, R=W.CS_R, T=W.CS_T_085)],
                     G=[[-1.0]], tau=[tau])
        s = make_oracle(wl, dict(rho=[_flat(nx, ny, W.CS_RHO_L_085, W.CS_RHO_V_085)]))
        s.step(6000)
        r = s.get_macroscopic()[0][0].reshape(ny, nx)[0]
        out.append((r[nx // 2], r[0]))
    assert abs(out[0][0] - out[1][0]) < 2e-4 * out[0][0]
    assert abs(out[0][1] - out[1][1]) < 5e-3 * out[0][1]


def test_exp_pseudopotential_density_ratio():
    """psi = exp(-1/rho) gives rho_l/rho_v ~ 7.6.  The paper does not print g; with g = -10/3
    (classic G = -10, reading R2) Maxwell's construction on p = c_s^2 rho + (g/2) psi^2 gives 7.57, and
    the simulated flat interface 7.05 (the EDM forcing error, same size as for CS above)."""
    g = -10.0 / 3.0
    pf = lambda r: r / 3 + 0.5 * g * np.exp(-2 / r)
    rr = np.linspace(0.05, 6, 200001)
    dp = np.diff(pf(rr))
    i1 = np.where((dp[:-1] > 0) & (dp[1:] <= 0))[0][0] + 1
    i2 = np.where((dp[:-1] < 0) & (dp[1:] >= 0))[0][0] + 1

    def area(ps):
        rv = brentq(lambda r: pf(r) - ps, 1e-3, rr[i1])
        rl = brentq(lambda r: pf(r) - ps, rr[i2], 50)
        v = np.linspace(1 / rl, 1 / rv, 100001)
        y = pf(1 / v) - ps
        return np.sum((y[1:] + y[:-1]) * np.diff(v)) / 2, rv, rl

    ps = brentq(lambda p: area(p)[0], max(pf(rr[i2]), 1e-9) + 1e-9, pf(rr[i1]) - 1e-9)
    _, rv, rl = area(ps)
    ratio_paper, tol = _scalars()["exp_psi_density_ratio"]
    assert abs(rl / rv - ratio_paper) < 0.1            # Maxwell ratio of this reading: 7.57
    nx, ny = 128, 2
    wl = base_wl("D2Q9", (nx, ny, 1), psi_kind=["EXP"], G=[[g]])
    s = make_oracle(wl, dict(rho=[_flat(nx, ny, rl, rv)]))
    s.step(8000)
    rho, _, p = s.get_macroscopic()
    r, pp = rho[0].reshape(ny, nx)[0], p.reshape(ny, nx)[0]
    assert abs(r[nx // 2] / r[0] - ratio_paper) < tol
    assert abs(r[nx // 2] / rl - 1) < 0.03 and abs(r[0] / rv - 1) < 0.12
    assert abs(pp[nx // 2] - pp[0]) < 2e-3 * pp[0]


def test_laplace_law():
    """Eq. 19: dp = sigma / R.  CS, T_r = 0.85, D2Q9: dp * R constant over the radii."""
    n = 64
    sig = []
    for R in (12, 16, 20):
        wl = base_wl("D2Q9", (n, n, 1), psi_kind=["CS"], eos=[dict(a=W.CS_A, b=W.CS_B, R=W.CS_R, T=W.CS_T_085)],
                     G=[[-1.0]])
        y, x = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
        c = (n - 1) / 2
        rho = W.tanh_profile(np.sqrt((x - c) ** 2 + (y - c) ** 2), R, 3.0, W.CS_RHO_L_085, W.CS_RHO_V_085)
        s = make_oracle(wl, dict(rho=[rho.reshape(-1)]))
        s.step(3000)
        r, u, p = s.get_macroscopic()
        r, p = r[0].reshape(n, n), p.reshape(n, n)
        row = r[n // 2]
        mid = 0.5 * (row.max() + row.min())
        xs = [i + (row[i] - mid) / (row[i] - row[i + 1]) for i in range(n - 1)
              if (row[i] - mid) * (row[i + 1] - mid) <= 0 and row[i] != row[i + 1]]
        Rm = (xs[-1] - xs[0]) / 2
        dp = p[n // 2, n // 2] - p[0, 0]
        assert dp > 0
        sig.append(dp * Rm)
        assert np.abs(u).max() < _scalars()["spurious_current_max"][0]
    sig = np.array(sig)
    assert np.abs(sig / sig.mean() - 1).max() < 0.03


def _meniscus(drho_b, nx=64, ny=26, wall=2, steps=4000):
    """Slug of component A between two flat plates (the wetting set-up of configs 2 and 4: SC93 psi, g_AB = 7/6,
    Delta rho on the other component B); returns a function row -> x of the right-hand A|B interface."""
    g = 3.5 / 3
    wl = base_wl("D2Q9", (nx, ny, 1), nc=2, psi_kind=["SC93"] * 2, eos=[dict(rho0=1.0)] * 2, G=[[0, g], [g, 0]],
                 wetting=[dict(phi=1, drho=0, lo=0, hi=1.2), dict(phi=1, drho=drho_b, lo=0, hi=1.2)])
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    mask = ((y < wall) | (y >= ny - wall)).astype(np.uint8)
    inA = (x >= nx // 4) & (x < 3 * nx // 4)
    a = np.where(inA, 1.0, 0.03)
    b = np.where(inA, 0.03, 1.0)
    s = make_oracle(wl, dict(rho=[a.reshape(-1), b.reshape(-1)], mask=mask.reshape(-1)))
    fluid = mask.reshape(-1) == 0
    m0 = [s.get_populations(k)[:, fluid].sum() for k in range(2)]
    s.step(steps)
    for k in range(2):
        assert abs(s.get_populations(k)[:, fluid].sum() - m0[k]) <= 1e-11 * m0[k]
    rho, _, _ = s.get_macroscopic()
    A, B = rho[0].reshape(ny, nx), rho[1].reshape(ny, nx)

    def cross(row):
        d = A[row] - B[row]
        for i in range(nx // 2, nx - 1):
            if d[i] > 0 and d[i + 1] <= 0:
                return i + d[i] / (d[i] - d[i + 1])
        raise AssertionError("no interface")

    return cross


def _contact_angle_circle_fit(drho_b, nx=64, ny=32, wall=2, steps=6000, skip=3):
    """Contact angle of component A from a least-squares circle through the interface points of all fluid rows but the
    `skip` next to each wall (centre on the channel axis): cos(theta) = (H/2) / R, H = plate distance (the walls sit
    half a cell outside the first / last fluid row)."""
    cross = _meniscus(drho_b, nx, ny, wall, steps)
    rows = np.arange(wall + skip, ny - wall - skip)
    xs = np.array([cross(int(r)) for r in rows])
    if np.ptp(xs) < 0.05:
        return 90.0
    yy = (rows - (ny - 1) / 2.0) ** 2
    # (x - xc)^2 + yy = R^2  ->  x^2 + yy = 2 xc x + (R^2 - xc^2)
    (xc, cc), *_ = np.linalg.lstsq(np.stack([2 * xs, np.ones_like(xs)], axis=1), xs ** 2 + yy, rcond=None)
    R = np.sqrt(cc + xc * xc)
    t = np.degrees(np.arccos(min(1.0, (ny - 2 * wall) / 2.0 / R)))
    return t if xs[len(xs) // 2] < xc else 180.0 - t      # centre of curvature on the B side: A wets


def _meniscus_offset(drho_b, nx=64, ny=26, wall=2, steps=4000):
    cross = _meniscus(drho_b, nx, ny, wall, steps)
    H = ny - 2 * wall
    dx = cross(wall) - cross(ny // 2)   # > 0: component A creeps along the wall (A wets)
    # circular meniscus: dx = (H/2)(1 - sin t)/cos t between the wall and the centre line
    t = np.degrees(np.pi / 2 - 2 * np.arctan(dx / (H / 2 - 0.5)))
    return dx, t


def test_contact_angle_neutral_and_monotone():
    """phi = 1, drho = 0 is neutral wetting (90 deg).  Lowering the virtual density of B at the
    wall (drho_B > 0, Eq. 17 second branch) makes A the wetting component; the angle falls monotonically."""
    angle, tol = _scalars()["neutral_contact_angle"]
    dx0, t0 = _meniscus_offset(0.0)
    assert abs(dx0) < 1e-6
    assert abs(t0 - angle) < tol
    dx1, t1 = _meniscus_offset(0.15)
    dx2, t2 = _meniscus_offset(0.30)
    assert 0 < dx1 < dx2
    assert angle > t1 > t2 > 30.0


def test_contact_angles_of_configs_2_and_4():
    """BASELINE.json: config 2 "wall virtual density set for a 60 deg contact angle", config 4 "a 40 deg contact angle for
    the wetting phase".  The Delta rho values workloads.py gives the two configs produce these angles (within 4 deg, the
    accuracy of a circle fit through a 3-cell-wide interface in a 28-cell channel).  Config 4 runs D3Q19; its
    z-invariant solutions are D2Q9 solutions (the D3Q19 weights project onto the D2Q9 ones: 1/18 + 2/36 = 1/9,
    1/3 + 2/18 = 4/9), so the flat-wall calibration is done in 2-D."""
    assert abs(_contact_angle_circle_fit(W.C2_DRHO_B) - 60.0) < 4.0
    assert abs(_contact_angle_circle_fit(W.C4_DRHO_NW) - 40.0) < 4.0
    wl2, _ = W.config2(32, 16)
    wl4, _ = W.config4(24)
    assert wl2["wetting"][1]["drho"] == W.C2_DRHO_B and wl2["wetting"][0]["drho"] == 0.0
    assert wl4["wetting"][0]["drho"] == W.C4_DRHO_NW and wl4["wetting"][1]["drho"] == 0.0


# ------------------------------------------------------------------ NEXT-1: A-weighted Zhang-Chen force (Eq. 11-13)
def _cs_wl(n, A, lattice="D2Q9", **kw):
    return base_wl(lattice, n, psi_kind=["CS"], eos=[dict(a=W.CS_A, b=W.CS_B, R=W.CS_R, T=W.CS_T_085)], G=[[-1.0]],
                   zc_A=[A], **kw)


@pytest.mark.parametrize("lattice,n", [("D2Q9", (64, 48, 1)), ("D3Q19", (40, 32, 24))])
def test_zhang_chen_force_is_minus_grad_U(lattice, n):
    """A = 1: F = F_ZC = -sum_i G_i U(x+e_i) e_i is a second-order approximation of -grad U with
    U = alpha p_EOS - c_s^2 rho (Eq. 11 first term, Eq. 12 second line); the EOS pressure is re-typed here."""
    d = 2 if lattice == "D2Q9" else 3
    z, y, x = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
    kx, ky = 2 * np.pi / n[0], 2 * np.pi / n[1]
    rho = 0.15 + 0.05 * np.sin(kx * x) * np.cos(ky * y)
    drx, dry = 0.05 * kx * np.cos(kx * x) * np.cos(ky * y), -0.05 * ky * np.sin(kx * x) * np.sin(ky * y)
    a, b, RT = W.CS_A, W.CS_B, W.CS_R * W.CS_T_085
    eta = lambda r: b * r / 4
    p = lambda r: r * RT * (1 + eta(r) + eta(r) ** 2 - eta(r) ** 3) / (1 - eta(r)) ** 3 - a * r * r
    h = 1e-6
    dU = ((p(rho + h) - p(rho - h)) / (2 * h) - 1.0 / 3.0)        # dU/drho
    s = make_oracle(_cs_wl(n, 1.0, lattice), dict(rho=[rho.reshape(-1)]))
    F = s.get_force(0)
    scale = np.abs(dU * drx).max()
    assert np.abs(F[0] + (dU * drx).reshape(-1)).max() < 0.03 * scale
    assert np.abs(F[1] + (dU * dry).reshape(-1)).max() < 0.03 * scale
    if d == 3:
        assert np.abs(F[2]).max() < 1e-15
    # A = 0 is the plain Shan-Chen force, A = 0.3 the weighted sum of the two (Eq. 13, first line)
    f0 = make_oracle(_cs_wl(n, 0.0, lattice), dict(rho=[rho.reshape(-1)])).get_force(0)
    f3 = make_oracle(_cs_wl(n, 0.3, lattice), dict(rho=[rho.reshape(-1)])).get_force(0)
    assert np.abs(f3 - (0.3 * F + 0.7 * f0)).max() < 1e-15
    # both forms discretise the same continuum force: -grad U = -g psi grad psi since U = g psi^2 / 2
    assert np.abs(F[0] - f0[0]).max() < 0.05 * scale


def test_zhang_chen_weight_brings_coexistence_to_maxwell_and_conserves():
    """the weighted force reaches densities the single schemes do not.  For CS at T_r = 0.85 a
    weight A ~ -0.19 brings the flat-interface vapour density from -8 % (A = 0, test above) to within 1.5 % of Maxwell's
    construction and keeps the liquid within 0.2 %.  Mass is conserved to rounding and total momentum stays zero
    (F_ZC sums to zero over a periodic box just as F_SC does)."""
    nx, ny = 128, 2
    s = make_oracle(_cs_wl((nx, ny, 1), -0.19), dict(rho=[_flat(nx, ny, W.CS_RHO_L_085, W.CS_RHO_V_085)]))
    m0 = s.get_macroscopic()[0][0].sum()
    s.step(8000)
    rho, u, p = s.get_macroscopic()
    r = rho[0].reshape(ny, nx)[0]
    assert abs(r[nx // 2] / W.CS_RHO_L_085 - 1) < 2e-3
    assert abs(r[0] / W.CS_RHO_V_085 - 1) < 1.5e-2
    assert abs(rho[0].sum() / m0 - 1) < 1e-12
    assert np.abs(s.get_force(0).sum(axis=1)).max() < 1e-12


# ------------------------------------------------------------------ NEXT-3: body force and cocurrent flow (Eq. 23)
def test_body_force_adds_mass_times_acceleration_per_step():
    """Periodic box, two components, interaction on: total momentum after t steps is t * (total mass) * a exactly
    (the interaction forces cancel pairwise, the body force is rho^k a on every cell)."""
    g = 0.4
    a = (1e-5, -2e-5, 3e-5)
    wl = base_wl("D3Q19", (12, 10, 8), nc=2, G=[[0.0, g], [g, 0.0]], tau=[0.8, 1.1], body_accel=a)
    rng = np.random.default_rng(3)
    rho = [0.5 + 0.2 * rng.uniform(size=960), 0.3 + 0.2 * rng.uniform(size=960)]
    s = make_oracle(wl, dict(rho=rho))
    mass = sum(r.sum() for r in rho)
    e, w, opp = o.lattice("D3Q19")
    t = 50
    s.step(t)
    mom = sum(s.get_populations(k).sum(axis=1) @ e for k in range(2))
    assert np.abs(mom - t * mass * np.array(a)).max() < 1e-11


def _channel(H, nx=4):
    m = np.zeros((H + 2, nx), dtype=np.uint8)
    m[0, :] = m[-1, :] = 1
    return m.reshape(-1)


def test_body_force_poiseuille_profile():
    """Plane channel of H fluid rows between halfway bounce-back walls, single component, no interaction: the steady
    Eq. 6 velocity is the parabola a/(2 nu) (y + 1/2)(H - 1/2 - y) (wall planes half a cell outside the fluid rows)."""
    H, nx, tau, acc = 24, 4, 0.9, 1e-6
    nu = (tau - 0.5) / 3.0
    wl = base_wl("D2Q9", (nx, H + 2, 1), tau=[tau], body_accel=(acc, 0.0, 0.0))
    s = make_oracle(wl, dict(rho=[np.ones(nx * (H + 2))], mask=_channel(H, nx)))
    s.step(int(6 * H * H / nu))
    u = s.get_macroscopic()[1][0].reshape(H + 2, nx)[1:-1, 0]
    y = np.arange(H)
    exact = acc / (2 * nu) * (y + 0.5) * (H - 0.5 - y)
    assert np.abs(u - exact).max() < 0.01 * exact.max()


def test_cocurrent_flow_relative_permeability_matches_eq23():
    """layered cocurrent flow of two components (psi = rho, g_intra = -0.027, g_inter = 0.57 as in
    P:275, both tau = 1 so M = 1), non-wetting in the centre, driven by a body force.  K_r of each phase = its flow
    rate over the flow rate of the whole channel run single-phase (Eq. 22); Eq. 23 with M = 1."""
    H, nx, acc = 64, 4, 2e-7
    gi, gx = -0.027, 0.57
    for half_width in (12, 20):
        wl = base_wl("D2Q9", (nx, H + 2, 1), nc=2, G=[[gi, gx], [gx, gi]], tau=[1.0, 1.0], body_accel=(acc, 0.0, 0.0))
        yy = np.repeat(np.arange(H + 2), nx)
        centre = np.abs(yy - (H + 1) / 2) < half_width
        rho_nw = np.where(centre, 1.0, 0.03)
        rho_w = np.where(centre, 0.03, 1.0)
        s = make_oracle(wl, dict(rho=[rho_nw, rho_w], mask=_channel(H, nx)))
        s.step(40000)
        rho, u, p = s.get_macroscopic()
        ux = u[0].reshape(H + 2, nx)[1:-1, 0]
        frac_nw = (rho[0] / (rho[0] + rho[1] + 1e-300)).reshape(H + 2, nx)[1:-1, 0]
        q_total_single = acc / (2 * (1.0 / 6.0)) * H ** 3 / 6.0      # integral of the single-phase parabola over the channel
        k_nw = (ux * frac_nw).sum() / q_total_single
        k_w = (ux * (1 - frac_nw)).sum() / q_total_single
        sw = 1.0 - frac_nw.sum() / H
        assert abs(k_w - 0.5 * sw ** 2 * (3 - sw)) < 0.02
        assert abs(k_nw - (1 - sw) * (1.5 + (1 - sw) ** 2 * (1 - 1.5))) < 0.02


# ------------------------------------------------------------------ NEXT-2: surface-tension control (Eq. 14-16, D2Q9 MRT)
def _droplet_sigma(kappa, A=0.0, R=16, n=64, steps=4000):
    wl = base_wl("D2Q9", (n, n, 1), psi_kind=["CS"], eos=[dict(a=W.CS_A, b=W.CS_B, R=W.CS_R, T=W.CS_T_085)], G=[[-1.0]],
                 collision="MRT", mrt_rates=[W.mrt_rates("D2Q9", 1.0)], st_kappa=[kappa], zc_A=[A])
    y, x = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    c = (n - 1) / 2
    rho = W.tanh_profile(np.sqrt((x - c) ** 2 + (y - c) ** 2), R, 3.0, W.CS_RHO_L_085, W.CS_RHO_V_085)
    s = make_oracle(wl, dict(rho=[rho.reshape(-1)]))
    s.step(steps)
    r, u, p = s.get_macroscopic()
    r, p = r[0].reshape(n, n), p.reshape(n, n)
    row = r[n // 2]
    mid = 0.5 * (row.max() + row.min())
    xs = [i + (row[i] - mid) / (row[i] - row[i + 1]) for i in range(n - 1)
          if (row[i] - mid) * (row[i + 1] - mid) <= 0 and row[i] != row[i + 1]]
    return (p[n // 2, n // 2] - p[0, 0]) * (xs[-1] - xs[0]) / 2, row.max(), row.min()


def test_surface_tension_scales_with_one_minus_kappa():
    """"the surface tension [scales] with 1 - kappa" while the mechanical stability (coexistence densities) is
    kept (Table 1: densities kappa-independent to ~0.7 %).  Laplace droplet, sigma = dp R."""
    s0, rl0, rv0 = _droplet_sigma(0.0)
    s5, rl5, rv5 = _droplet_sigma(0.5)
    assert abs(s5 / s0 - 0.5) < 0.04
    assert abs(rl5 / rl0 - 1) < 5e-3 and abs(rv5 / rv0 - 1) < 3e-2
