"""Pins for single terms of the oracle that the physics tests only see through loose tolerances (CPU only).

Every check is exact (rounding level) or a paper value, and is chosen so that ONE plausible mistake in
oracle/lbm_oracle.cpp fails it:
  * velocity-shift forcing at tau != 1 (reading R7, cited P:121)      -> momentum gain per step = total force
  * the w_i weights of rho_ave in Eq. 17 (reading R11/R12)  -> hand-built non-uniform neighbourhood
  * the 1/2 F of Eq. 6                                          -> u = (t + 1/2) a in a uniform fluid
  * D3Q19 MRT rate <-> moment-row assignment (reading R9)        -> shear-wave viscosity on axes and diagonals
  * source C and tensor Q of Eq. 15-16 incl. the A_kk term -> domain-summed moments after one step,
    and the sigma(kappa) ratios of the paper's Table 2
  * O(u^2) terms of the pressure face (reading R10)      -> uniform equilibrium flow is a fixed point
"""
from pathlib import Path

import numpy as np
import pytest

from conftest import make_oracle
from oracle import lbm_oracle as o
from paper_2506_17713_b200 import workloads as W
from test_oracle_basics import base_wl

GOLD = Path(__file__).parent / "golden"


# ------------------------------------------------------------------ (a) velocity shift at tau != 1  (R7)
@pytest.mark.parametrize("collision", ["BGK", "MRT"])
def test_shift_forcing_momentum_gain_is_total_force(collision):
    """With u_eq^k = u' + tau_k F^k/rho^k and the common velocity u' (R6) the momentum gained in one collision is
    sum_k [rho^k u'/tau_k - j^k/tau_k] + sum_k F^k = sum_k F^k.  On a periodic box the interaction forces cancel in
    pairs and the body force is rho^k a, so after t steps the total momentum is t * mass * a EXACTLY.
    (`u_eq = u' + F/rho` would gain sum_k F^k/tau_k instead: 1.25 / 0.91 times too much / little here.)"""
    g = 0.4
    a = (1e-5, -2e-5, 3e-5)
    tau = [0.8, 1.1]
    kw = {}
    if collision == "MRT":
        kw = dict(collision="MRT", mrt_rates=[W.mrt_rates("D3Q19", tau[0]), W.mrt_rates("D3Q19", tau[1])])
    wl = base_wl("D3Q19", (12, 10, 8), nc=2, G=[[0.0, g], [g, 0.0]], tau=tau, body_accel=a, forcing="SHIFT", **kw)
    rng = np.random.default_rng(31)
    rho = [0.5 + 0.2 * rng.uniform(size=960), 0.3 + 0.2 * rng.uniform(size=960)]
    s = make_oracle(wl, dict(rho=rho))
    mass = sum(r.sum() for r in rho)
    e, _, _ = o.lattice("D3Q19")
    for t in (1, 40):
        s.step(t if t == 1 else t - 1)
        mom = sum(s.get_populations(k).sum(axis=1) @ e for k in range(2))
        assert np.abs(mom - t * mass * np.array(a)).max() < 1e-12, (t, mom)


# ------------------------------------------------------------------ (b) rho_ave weights of Eq. 17
@pytest.mark.parametrize("lattice,n", [("D2Q9", (7, 6, 1)), ("D3Q19", (6, 5, 5))])
def test_virtual_density_weights_on_a_non_uniform_neighbourhood(lattice, n):
    """One boundary solid whose neighbours all carry different densities, some of them solid too:
    rho_s = clamp(phi * sum_i w_i rho(x+e_i)[fluid] / sum_i w_i [fluid] - drho, lo, hi) with the LATTICE weights
    (axis 1/9 | 1/18, diagonal 1/36) typed here.  Equal weights, or a sum over all neighbours, give another number."""
    nx, ny, nz = n
    N = nx * ny * nz
    rng = np.random.default_rng(17)
    rho = [rng.uniform(0.2, 1.4, N), rng.uniform(0.05, 0.9, N)]
    mask = np.zeros((nz, ny, nx), np.uint8)
    c = (2, 2, 2 if nz > 1 else 0)
    mask[c[2], c[1], c[0]] = 1
    mask[c[2], c[1], c[0] + 1] = 1            # +x neighbour solid
    mask[c[2], c[1] - 1, c[0] - 1] = 1        # (-1,-1,0) neighbour solid
    if nz > 1:
        mask[c[2] + 1, c[1], c[0]] = 1        # +z neighbour solid
    wet = [dict(phi=1.3, drho=0.0, lo=0.0, hi=10.0), dict(phi=1.0, drho=0.07, lo=0.0, hi=10.0)]
    wl = base_wl(lattice, n, nc=2, G=[[0.0, 0.3], [0.3, 0.0]], wetting=wet)
    s = make_oracle(wl, dict(rho=rho, mask=mask.reshape(-1)))
    got, _, _ = s.get_macroscopic()
    w_axis = 1.0 / 9.0 if lattice == "D2Q9" else 1.0 / 18.0
    w_diag = 1.0 / 36.0
    for k in range(2):
        f = rho[k].reshape(nz, ny, nx)
        num = den = 0.0
        for dz in ((-1, 0, 1) if nz > 1 else (0,)):
            for dy in (-1, 0, 1):
                for dx in (-1, 0, 1):
                    m2 = dx * dx + dy * dy + dz * dz
                    if m2 == 0 or m2 == 3:
                        continue
                    z, y, x = (c[2] + dz) % nz, (c[1] + dy) % ny, (c[0] + dx) % nx
                    if mask[z, y, x]:
                        continue
                    w = w_axis if m2 == 1 else w_diag
                    num += w * f[z, y, x]
                    den += w
        expect = wet[k]["phi"] * num / den - wet[k]["drho"]
        idx = c[0] + nx * (c[1] + ny * c[2])
        assert abs(got[k][idx] - expect) < 1e-14, (k, got[k][idx], expect)
        # unweighted mean over the same fluid neighbours is measurably different (the test has teeth)
        plain = np.mean([f[(c[2] + dz) % nz, (c[1] + dy) % ny, (c[0] + dx) % nx]
                         for dz in ((-1, 0, 1) if nz > 1 else (0,)) for dy in (-1, 0, 1) for dx in (-1, 0, 1)
                         if 0 < dx * dx + dy * dy + dz * dz < 3 and not mask[(c[2] + dz) % nz, (c[1] + dy) % ny, (c[0] + dx) % nx]])
        assert abs(wet[k]["phi"] * plain - wet[k]["drho"] - expect) > 1e-3
    # limiter: the same cell with tight bounds is clamped
    wet2 = [dict(phi=1.3, drho=0.0, lo=0.0, hi=0.31), dict(phi=1.0, drho=0.07, lo=0.66, hi=10.0)]
    s2 = make_oracle(dict(wl, wetting=wet2), dict(rho=rho, mask=mask.reshape(-1)))
    got2, _, _ = s2.get_macroscopic()
    idx = c[0] + nx * (c[1] + ny * c[2])
    assert got2[0][idx] == pytest.approx(min(got[0][idx], 0.31), abs=0) and got2[1][idx] == pytest.approx(max(got[1][idx], 0.66), abs=0)
    # solids without a fluid neighbour would keep rho = 0; here every solid touches fluid, so all four are listed
    assert len(s.get_boundary_solids()) == int(mask.sum())


# ------------------------------------------------------------------ (c) Eq. 6: half-force velocity
@pytest.mark.parametrize("lattice,n,forcing", [("D2Q9", (6, 5, 1), "EDM"), ("D3Q19", (5, 4, 3), "EDM"), ("D2Q9", (6, 5, 1), "SHIFT")])
def test_output_velocity_carries_half_the_force(lattice, n, forcing):
    """Uniform fluid at rest, uniform body force, periodic: every step adds rho a to j, so j(t) = t rho a and the
    exported velocity of Eq. 6 is u = (j + F/2)/rho = (t + 1/2) a exactly (tau-independent for both schemes)."""
    a = np.array([3e-5, -1e-5, 2e-5 if lattice == "D3Q19" else 0.0])
    d = 2 if lattice == "D2Q9" else 3
    N = n[0] * n[1] * n[2]
    wl = base_wl(lattice, n, tau=[0.7], forcing=forcing, body_accel=tuple(a), G=[[-0.3]])
    s = make_oracle(wl, dict(rho=[np.full(N, 0.8)]))
    for t in (0, 1, 7):
        if t:
            s.step(1 if t == 1 else 6)
        _, u, _ = s.get_macroscopic()
        assert np.abs(u - ((t + 0.5) * a[:d])[:, None]).max() < 1e-16 + 1e-13 * np.abs(a).max(), t


# ------------------------------------------------------------------ (d) D3Q19 MRT: which row carries which rate  (R9)
_WAVES = [  # (velocity direction, wave vector direction): transverse waves on the axes and on the face diagonals
    ((1, 0, 0), (0, 1, 0)), ((0, 1, 0), (0, 0, 1)), ((0, 0, 1), (1, 0, 0)),      # p_xy, p_yz, p_xz
    ((1, 1, 0), (1, -1, 0)), ((0, 1, 1), (0, 1, -1)), ((1, 0, 1), (1, 0, -1)),   # p_xx - p_yy, p_yy - p_zz, p_xx - p_zz
]


@pytest.mark.parametrize("vel,wave", _WAVES)
def test_d3q19_mrt_shear_viscosity_with_config3_rates(vel, wave):
    """nu = c_s^2 (1/s_nu - 1/2) for the rates workloads.mrt_rates feeds to BOTH sides (config 3's, at tau = 0.8 so
    that s_nu = 1.25 differs from every other rate: 1.19, 1.4, 1.2, 1.98).  Six transverse shear waves reach all five
    stress moments (rows 9, 11, 13, 14, 15 of the d'Humieres basis); a rate put on a neighbouring row (e.g. s_pi = 1.4
    on row 9) changes nu by 29 %."""
    n = 24
    tau = 0.8
    wl = base_wl("D3Q19", (n, n, n), tau=[tau], collision="MRT", mrt_rates=[W.mrt_rates("D3Q19", tau)])
    z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    k0 = 2 * np.pi / n
    phase = k0 * (wave[0] * x + wave[1] * y + wave[2] * z)
    k2 = k0 * k0 * sum(c * c for c in wave)
    vhat = np.array(vel, float) / np.sqrt(sum(c * c for c in vel))
    U = 1e-3
    u = (vhat[:, None] * (U * np.sin(phase)).reshape(1, -1))
    s = make_oracle(wl, dict(rho=[np.ones(n ** 3)], u=u))
    T = 120
    s.step(T)
    _, uu, _ = s.get_macroscopic()
    amp = 2 * np.mean((vhat @ uu) * np.sin(phase).reshape(-1))
    nu_meas = -np.log(amp / U) / (k2 * T)
    nu = (tau - 0.5) / 3.0
    assert abs(nu_meas - nu) / nu < 0.02, (nu_meas, nu)


# ------------------------------------------------------------------ (e) Eq. 15-16 incl. the A_kk term
def _gold_table2():
    out = {}
    for line in (GOLD / "table2_surface_tension.txt").read_text().splitlines():
        if line and not line.startswith("#"):
            p = line.split()
            out[p[0]] = [float(v) for v in p[1:]]
    return out


@pytest.mark.parametrize("A", [0.0, -0.19, 0.35])
def test_surface_tension_source_moments_after_one_step(A):
    """Eq. 14-16 with reading R20.  Streaming permutes the populations of a periodic box, so the domain
    sum of a moment after one step is the domain sum of its post-collision value; between a run with kappa and a run
    without, the moments of f* differ by exactly C (M M^-1 C = C).  Hence
        sum_x [m_r(kappa) - m_r(0)] = sum_x C_r(x),   r = 0..8,
    with C of Eq. 15 and Q of Eq. 16 evaluated here with numpy on the psi field (times g_kk, R20).  Pins the entries
    and signs of C, their rates, the e e weighting, and the (A/2)(psi'^2 - psi^2) term."""
    n = (16, 12, 1)
    N = n[0] * n[1]
    rates = W.mrt_rates("D2Q9", 0.9)
    kappa, g = 0.4, -1.0
    common = dict(psi_kind=["CS"], eos=[dict(a=W.CS_A, b=W.CS_B, R=W.CS_R, T=W.CS_T_085)], G=[[g]], collision="MRT",
                  mrt_rates=[rates], tau=[0.9], zc_A=[A])
    rng = np.random.default_rng(23)
    rho = rng.uniform(0.05, 0.3, N)
    s1 = make_oracle(base_wl("D2Q9", n, st_kappa=[kappa], **common), dict(rho=[rho]))
    s0 = make_oracle(base_wl("D2Q9", n, st_kappa=[0.0], **common), dict(rho=[rho]))
    psi = s0.get_psi(0).reshape(n[1], n[0])
    s1.step(1)
    s0.step(1)
    M, _ = o.mrt_matrices("D2Q9")
    dm = M @ (s1.get_populations(0) - s0.get_populations(0)).sum(axis=1)
    e, w, _ = o.lattice("D2Q9")
    Q = np.zeros((2, 2))
    for i in range(1, 9):
        ps1 = np.roll(psi, (-e[i][1], -e[i][0]), axis=(0, 1))          # psi(x + e_i)
        t = 3.0 * w[i] * ((1 - A) * psi * (ps1 - psi) + 0.5 * A * (ps1 ** 2 - psi ** 2))
        Q += kappa * g * t.sum() * np.outer(e[i][:2], e[i][:2])
    C = np.zeros(9)
    C[1] = 1.5 * rates[1] * (Q[0, 0] + Q[1, 1])
    C[2] = -1.5 * rates[2] * (Q[0, 0] + Q[1, 1])
    C[7] = -rates[7] * (Q[0, 0] - Q[1, 1])
    C[8] = -rates[8] * Q[0, 1]
    assert np.abs(C[[1, 2, 7, 8]]).min() > 1e-5          # every entry is exercised
    assert np.abs(dm - C).max() < 1e-13, (dm, C)


@pytest.mark.parametrize("A", [0.0, -0.19])
def test_surface_tension_ratio_matches_paper_table2(A):
    """Table 2, Carnahan-Starling row: sigma = 0.0186 / 0.0085 at 1 - kappa = 1.0 / 0.5, i.e. a ratio
    0.457 (the absolute values need the paper's unpublished alpha, A and T_r = 0.8 MRT set-up; the RATIO is what
    Eq. 16's normalisation fixes).  With R20 (factor g_kk, no 1/2) the Laplace-droplet ratio is 0.47 at A = 0 and
    0.42 at A = -0.19; Li & Luo's original kappa G/2 would give 0.73.  The slope is steeper than 1 - kappa because the
    exact-difference forcing adds its own F F / rho term to the pressure tensor (R20)."""
    from test_oracle_physics import _droplet_sigma
    cs = _gold_table2()["CS"]
    paper_ratio = cs[1] / cs[0]
    s0, _, _ = _droplet_sigma(0.0, A)
    s5, rl5, rv5 = _droplet_sigma(0.5, A)
    assert abs(s5 / s0 - paper_ratio) < 0.04, (s5 / s0, paper_ratio)


# ------------------------------------------------------------------ (f) pressure face, O(u^2) terms  (R10)
@pytest.mark.parametrize("lattice,n", [("D2Q9", (9, 6, 1)), ("D3Q19", (7, 5, 4))])
def test_pressure_faces_pass_uniform_equilibrium_flow_exactly(lattice, n):
    """f_eq,i + f_eq,ibar = 2 w_i rho [1 + (e_i.u)^2/(2 c_s^4) - u^2/(2 c_s^2)] identically, so with anti-bounce-back
    faces at density rho_w on both ends a uniform equilibrium flow (rho_w, u0) at ANY Mach number is a fixed point of
    the step, if and only if the O(u^2) bracket of reading R10 is exactly this one, evaluated with the node's own
    velocity.  Dropping either quadratic term, or a wrong coefficient, moves f by ~ w rho u^2 = 1e-4 per step."""
    d = 2 if lattice == "D2Q9" else 3
    N = n[0] * n[1] * n[2]
    rho_w = 0.9
    u0 = np.array([0.08, 0.03, -0.02 if d == 3 else 0.0])
    wl = base_wl(lattice, n, periodic=(False, True, True), tau=[0.8],
                 face_bc={0: ("PRESSURE", (rho_w,), (0, 0, 0)), 1: ("PRESSURE", (rho_w,), (0, 0, 0))})
    u = np.repeat(u0[:d, None], N, axis=1)
    s = make_oracle(wl, dict(rho=[np.full(N, rho_w)], u=u))
    f0 = s.get_populations(0)
    assert np.abs(f0 - o.feq(lattice, rho_w, u0)[:, None]).max() < 1e-16
    s.step(25)
    assert np.abs(s.get_populations(0) - f0).max() < 1e-14
    # teeth: the same run with a face density 1 % off is visibly not a fixed point
    wl2 = dict(wl, face_bc={0: ("PRESSURE", (1.01 * rho_w,), (0, 0, 0)), 1: ("PRESSURE", (rho_w,), (0, 0, 0))})
    s2 = make_oracle(wl2, dict(rho=[np.full(N, rho_w)], u=u))
    s2.step(1)
    assert np.abs(s2.get_populations(0) - f0).max() > 1e-4
