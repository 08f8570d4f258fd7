"""Pins for the oracle's building blocks (CPU only).

Each test holds oracle/lbm_oracle.cpp to something other than itself: closed
forms, conservation laws, textbook limits, library routines (numpy float16,
np.roll), or values from tests/golden/ (each with its citation).
"""
from pathlib import Path

import numpy as np
import pytest

from conftest import make_oracle
from oracle import lbm_oracle as o

GOLD = Path(__file__).parent / "golden"


def base_wl(lattice="D2Q9", n=(16, 12, 1), nc=1, **kw):
    wl = dict(lattice=lattice, nx=n[0], ny=n[1], nz=n[2], n_components=nc, periodic=(True, True, True),
              psi_kind=["RHO"] * nc, eos=[dict()] * nc, G=[[0.0] * nc for _ in range(nc)],
              collision="BGK", tau=[1.0] * nc, forcing="EDM", compute_dtype="f64", store_dtype="f64")
    wl.update(kw)
    return wl


# ------------------------------------------------------------------ lattice (R1)
@pytest.mark.parametrize("name,q,d", [("D2Q9", 9, 2), ("D3Q19", 19, 3)])
def test_lattice_isotropy(name, q, d):
    e, w, opp = o.lattice(name)
    assert e.shape == (q, 3)
    cs2 = 1.0 / 3.0
    assert abs(w.sum() - 1) < 1e-15
    assert np.allclose((w[:, None] * e).sum(0), 0, atol=1e-16)
    second = np.einsum("i,ia,ib->ab", w, e, e)[:d, :d]
    assert np.allclose(second, cs2 * np.eye(d), atol=1e-15)
    third = np.einsum("i,ia,ib,ic->abc", w, e, e, e)
    assert np.allclose(third, 0, atol=1e-16)
    fourth = np.einsum("i,ia,ib,ic,id->abcd", w, e, e, e, e)[:d, :d, :d, :d]
    I = np.eye(d)
    iso = cs2 * cs2 * (np.einsum("ab,cd->abcd", I, I) + np.einsum("ac,bd->abcd", I, I) + np.einsum("ad,bc->abcd", I, I))
    assert np.allclose(fourth, iso, atol=1e-15)
    assert np.all(e[opp] == -e)
    assert len({tuple(v) for v in e}) == q  # distinct velocities
    assert np.all(e[0] == 0)


# ------------------------------------------------------------------ f_eq moments
@pytest.mark.parametrize("name,d", [("D2Q9", 2), ("D3Q19", 3)])
def test_feq_moments_closed_form(name, d):
    e, w, _ = o.lattice(name)
    rng = np.random.default_rng(0)
    for _ in range(20):
        rho = rng.uniform(0.01, 9.0)
        u = np.zeros(3)
        u[:d] = rng.uniform(-0.15, 0.15, size=d)
        f = o.feq(name, rho, u)
        assert abs(f.sum() - rho) <= 2e-15 * rho
        mom = (f[:, None] * e).sum(0)
        assert np.allclose(mom, rho * u, rtol=0, atol=3e-15 * rho)
        P = np.einsum("i,ia,ib->ab", f, e, e)[:d, :d]
        assert np.allclose(P, rho * (np.eye(d) / 3.0 + np.outer(u[:d], u[:d])), rtol=0, atol=4e-15 * rho)
    # rest state: f_eq = w rho
    assert np.allclose(o.feq(name, 2.0, [0, 0, 0]), 2.0 * w, rtol=0, atol=1e-16)


# ------------------------------------------------------------------ MRT basis (R9)
@pytest.mark.parametrize("name", ["D2Q9", "D3Q19"])
def test_mrt_basis(name):
    M, Mi = o.mrt_matrices(name)
    e, w, _ = o.lattice(name)
    q = len(w)
    gold = {}
    for line in (GOLD / "mrt_row_norms.txt").read_text().splitlines():
        if line and not line.startswith("#"):
            parts = line.split()
            gold[parts[0]] = np.array([float(v) for v in parts[1:]])
    gram = M @ M.T
    assert np.allclose(gram - np.diag(np.diag(gram)), 0, atol=1e-12)  # rows orthogonal
    assert np.allclose(np.diag(gram), gold[name])
    assert np.allclose(Mi @ M, np.eye(q), atol=1e-14)
    # conserved rows: density and momentum
    assert np.allclose(M[0], 1)
    jrows = [3, 5] if name == "D2Q9" else [3, 5, 7]
    for a, r in enumerate(jrows):
        assert np.allclose(M[r], e[:, a])
    # integer entries
    assert np.allclose(M, np.round(M))
    # stress rows annihilate the isotropic part: M_stress . w = 0
    srows = [7, 8] if name == "D2Q9" else [9, 11, 13, 14, 15]
    assert np.allclose(M[srows] @ w, 0, atol=1e-15)


def test_d3q19_equilibrium_moments_closed_form():
    """m_eq = M f_eq (Eq. 3 taken literally, R9) has the textbook closed form of d'Humieres et al. (2002) with the
    second-order f_eq: e = -11 rho + 19 rho u^2, eps = 3 rho - 11/2 rho u^2, q = -2/3 j, 3 p_xx = rho (2 ux^2 - uy^2 - uz^2),
    3 pi_xx = -1/2 * 3 p_xx, p_ww = rho (uy^2 - uz^2), pi_ww = -1/2 p_ww, p_xy = rho ux uy, ..., m = 0.  Pins the row order
    and the signs of the oracle's D3Q19 basis (and the expressions the CUDA path evaluates instead of the product)."""
    M, _ = o.mrt_matrices("D3Q19")
    rng = np.random.default_rng(12)
    for _ in range(10):
        rho = rng.uniform(0.05, 8.0)
        ux, uy, uz = rng.uniform(-0.12, 0.12, 3)
        uu = ux * ux + uy * uy + uz * uz
        pxx, pww = rho * (2 * ux * ux - uy * uy - uz * uz), rho * (uy * uy - uz * uz)
        expect = np.array([rho, rho * (19 * uu - 11), rho * (3 - 5.5 * uu), rho * ux, -2 / 3 * rho * ux, rho * uy, -2 / 3 * rho * uy,
                           rho * uz, -2 / 3 * rho * uz, pxx, -0.5 * pxx, pww, -0.5 * pww, rho * ux * uy, rho * uy * uz, rho * ux * uz,
                           0, 0, 0])
        assert np.abs(M @ o.feq("D3Q19", rho, [ux, uy, uz]) - expect).max() < 1e-14 * rho * 30


# ------------------------------------------------------------------ fp16 storage rounding (R16)
def test_round_to_half_matches_numpy_float16():
    rng = np.random.default_rng(1)
    vals = np.concatenate([
        rng.uniform(-2, 2, 2000), rng.uniform(-1e-4, 1e-4, 2000), rng.uniform(-7e-8, 7e-8, 500),
        rng.uniform(-70000, 70000, 500),
        np.array([0.0, 1.0, 1.0 + 2 ** -11, 1.0 + 3 * 2 ** -11, 65504.0, 65519.9, 65520.0, 2 ** -14, 2 ** -24,
                  2 ** -25, 3 * 2 ** -25, 6.1e-5, 5.96e-8]),
    ]).astype(np.float32)
    with np.errstate(over="ignore"):
        ref = vals.astype(np.float16).astype(np.float32)
    got = np.array([o.round_to_half(float(v)) for v in vals], dtype=np.float32)
    assert np.array_equal(got, ref)


# ------------------------------------------------------------------ pure streaming = permutation
@pytest.mark.parametrize("lattice,n", [("D2Q9", (7, 5, 1)), ("D3Q19", (5, 4, 3))])
def test_pure_streaming_is_shift(lattice, n):
    wl = base_wl(lattice, n, no_collide=True)
    N = n[0] * n[1] * n[2]
    s = o.Oracle(wl)
    s.init_fields([np.ones(N)])
    e, w, _ = o.lattice(lattice)
    q = len(w)
    rng = np.random.default_rng(2)
    f0 = rng.uniform(0.1, 1.0, size=(q, N))
    s.set_populations(0, f0)
    steps = 3
    s.step(steps)
    f = s.get_populations(0).reshape(q, n[2], n[1], n[0])
    ref = f0.reshape(q, n[2], n[1], n[0]).copy()
    for i in range(q):
        ref[i] = np.roll(ref[i], shift=(steps * e[i, 2], steps * e[i, 1], steps * e[i, 0]), axis=(0, 1, 2))
    assert np.array_equal(f, ref)
    s.step(int(np.lcm.reduce(n)) - steps)
    assert np.array_equal(s.get_populations(0), f0)


# ------------------------------------------------------------------ conservation laws
def _momentum(s, lattice):
    e, _, _ = o.lattice(lattice)
    tot = np.zeros(3)
    for k in range(s.nc):
        f = s.get_populations(k)
        tot += (f.sum(1)[:, None] * e).sum(0)
    return tot


@pytest.mark.parametrize("lattice,n", [("D2Q9", (24, 20, 1)), ("D3Q19", (10, 8, 6))])
def test_conservation_single_component_cs(lattice, n):
    wl = base_wl(lattice, n, psi_kind=["CS"], eos=[dict(a=1.0, b=4.0, R=1.0, T=0.0802)], G=[[-1.0]])
    N = n[0] * n[1] * n[2]
    rng = np.random.default_rng(3)
    rho0 = 0.15 + 0.05 * rng.uniform(-1, 1, N)
    s = make_oracle(wl, dict(rho=[rho0]))
    m0 = s.get_populations(0).sum()
    s.step(200)
    m1 = s.get_populations(0).sum()
    assert abs(m1 - m0) <= 1e-12 * m0
    assert np.abs(_momentum(s, lattice)).max() <= 1e-11
    # the field actually evolved (phase separation under way)
    assert np.abs(s.get_macroscopic()[0][0] - rho0).max() > 1e-3


def test_conservation_two_components():
    n = (20, 16, 1)
    N = n[0] * n[1]
    g = 3.5 / 3
    wl = base_wl("D2Q9", n, nc=2, psi_kind=["SC93", "SC93"], eos=[dict(rho0=1.0)] * 2, G=[[0, g], [g, 0]], tau=[1.0, 0.8])
    rng = np.random.default_rng(4)
    a = 0.5 + 0.3 * rng.uniform(-1, 1, N)
    b = 0.5 + 0.3 * rng.uniform(-1, 1, N)
    s = make_oracle(wl, dict(rho=[a, b]))
    ma, mb = s.get_populations(0).sum(), s.get_populations(1).sum()
    s.step(300)
    assert abs(s.get_populations(0).sum() - ma) <= 1e-12 * ma
    assert abs(s.get_populations(1).sum() - mb) <= 1e-12 * mb
    assert np.abs(_momentum(s, "D2Q9")).max() <= 1e-11


# ------------------------------------------------------------------ collision-model identities
@pytest.mark.parametrize("lattice,n", [("D2Q9", (16, 12, 1)), ("D3Q19", (8, 6, 5))])
@pytest.mark.parametrize("tau", [1.0, 0.8])
def test_mrt_with_equal_rates_is_bgk(lattice, n, tau):
    q = 9 if lattice == "D2Q9" else 19
    N = n[0] * n[1] * n[2]
    rng = np.random.default_rng(5)
    rho0 = 0.15 + 0.05 * rng.uniform(-1, 1, N)
    kw = dict(psi_kind=["CS"], eos=[dict(a=1.0, b=4.0, R=1.0, T=0.0802)], G=[[-1.0]], tau=[tau])
    a = make_oracle(base_wl(lattice, n, **kw), dict(rho=[rho0]))
    b = make_oracle(base_wl(lattice, n, collision="MRT", mrt_rates=[[1.0 / tau] * q], **kw), dict(rho=[rho0]))
    a.step(50)
    b.step(50)
    assert np.abs(a.get_populations(0) - b.get_populations(0)).max() <= 1e-13


def test_edm_equals_shift_at_tau_one_and_differs_otherwise():
    n = (24, 16, 1)
    N = n[0] * n[1]
    rng = np.random.default_rng(6)
    rho0 = 0.15 + 0.05 * rng.uniform(-1, 1, N)
    kw = dict(psi_kind=["CS"], eos=[dict(a=1.0, b=4.0, R=1.0, T=0.0802)], G=[[-1.0]])
    out = {}
    for tau in (1.0, 0.8):
        for forcing in ("EDM", "SHIFT"):
            s = make_oracle(base_wl("D2Q9", n, tau=[tau], forcing=forcing, **kw), dict(rho=[rho0]))
            s.step(60)
            out[(tau, forcing)] = s.get_populations(0)
    assert np.abs(out[(1.0, "EDM")] - out[(1.0, "SHIFT")]).max() <= 1e-13
    assert np.abs(out[(0.8, "EDM")] - out[(0.8, "SHIFT")]).max() > 1e-7


# ------------------------------------------------------------------ viscosity: nu = c_s^2 (tau - 1/2)
@pytest.mark.parametrize("collision,tau", [("BGK", 0.8), ("BGK", 1.3), ("MRT", 0.8)])
def test_shear_wave_decay_gives_viscosity(collision, tau):
    """Textbook pin on collision + streaming: a shear wave u_x = U sin(k y) decays as exp(-nu k^2 t)."""
    nx, ny = 4, 48
    N = nx * ny
    kw = {}
    if collision == "MRT":
        from paper_2506_17713_b200.workloads import mrt_rates
        kw = dict(collision="MRT", mrt_rates=[mrt_rates("D2Q9", tau)])
    wl = base_wl("D2Q9", (nx, ny, 1), tau=[tau], **kw)
    y = np.repeat(np.arange(ny), nx).astype(float)
    k = 2 * np.pi / ny
    U = 1e-3
    u = np.zeros((2, N))
    u[0] = U * np.sin(k * y)
    s = make_oracle(wl, dict(rho=[np.ones(N)], u=u))
    T = 400
    s.step(T)
    _, uu, _ = s.get_macroscopic()
    amp = 2 * np.mean(uu[0] * np.sin(k * y))
    nu_meas = -np.log(amp / U) / (k * k * T)
    nu = (tau - 0.5) / 3.0
    assert abs(nu_meas - nu) / nu < 5e-3


# ------------------------------------------------------------------ force: continuum limit & normalisation (R2)
@pytest.mark.parametrize("lattice,n", [("D2Q9", (64, 48, 1)), ("D3Q19", (48, 40, 32))])
def test_force_is_minus_g_psi_grad_psi(lattice, n):
    """With G(x,x') = w_i/c_s^2 (sum G e e = I) Eq. 13's F_SC is a second-order
    approximation of Eq. 11's -g psi grad psi."""
    g = -0.7
    wl = base_wl(lattice, n, G=[[g]])
    d = 2 if lattice == "D2Q9" else 3
    z, y, x = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
    kx, ky, kz = 2 * np.pi / n[0], 2 * np.pi / n[1], 2 * np.pi / n[2]
    rho = 1.0 + 0.2 * np.sin(kx * x) * np.cos(ky * y) * (np.cos(kz * z) if d == 3 else 1.0)
    s = make_oracle(wl, dict(rho=[rho.reshape(-1)]))
    F = s.get_force(0)
    gx = 0.2 * kx * np.cos(kx * x) * np.cos(ky * y) * (np.cos(kz * z) if d == 3 else 1.0)
    gy = -0.2 * ky * np.sin(kx * x) * np.sin(ky * y) * (np.cos(kz * z) if d == 3 else 1.0)
    exact = [-g * rho * gx, -g * rho * gy]
    if d == 3:
        exact.append(-g * rho * (-0.2 * kz * np.sin(kx * x) * np.cos(ky * y) * np.sin(kz * z)))
    scale = abs(g) * 0.2 * kx
    for a in range(d):
        err = np.abs(F[a] - exact[a].reshape(-1)).max()
        assert err < 0.025 * scale, (a, err, scale)   # O(k^2) truncation error, ~|k|^2/6 relative
    # a uniform field exerts no force
    s2 = make_oracle(wl, dict(rho=[np.full(n[0] * n[1] * n[2], 0.7)]))
    assert np.abs(s2.get_force(0)).max() < 1e-15


# ------------------------------------------------------------------ walls: halfway bounce-back (R13)
def _box_mask(nx, ny, nz=1):
    m = np.zeros((nz, ny, nx), dtype=np.uint8)
    m[:, 0, :] = m[:, -1, :] = 1
    m[:, :, 0] = m[:, :, -1] = 1
    if nz > 1:
        m[0] = m[-1] = 1
    return m.reshape(-1)


@pytest.mark.parametrize("lattice,n", [("D2Q9", (18, 14, 1)), ("D3Q19", (10, 9, 8))])
def test_closed_box_conserves_mass(lattice, n):
    N = n[0] * n[1] * n[2]
    g = 3.5 / 3
    wl = base_wl(lattice, n, nc=2, psi_kind=["SC93", "SC93"], eos=[dict(rho0=1.0)] * 2, G=[[0, g], [g, 0]],
                 wetting=[dict(phi=1.0, drho=0.0, lo=0, hi=1.2), dict(phi=1.0, drho=0.2, lo=0, hi=1.2)])
    mask = _box_mask(*n)
    rng = np.random.default_rng(7)
    a = 0.5 + 0.4 * rng.uniform(-1, 1, N)
    b = 0.5 + 0.4 * rng.uniform(-1, 1, N)
    s = make_oracle(wl, dict(rho=[a, b], mask=mask))
    fluid = mask == 0
    m0 = [s.get_populations(k)[:, fluid].sum() for k in range(2)]
    s.step(200)
    for k in range(2):
        m1 = s.get_populations(k)[:, fluid].sum()
        assert abs(m1 - m0[k]) <= 1e-12 * m0[k]
    # solid cells are inert: still f_eq(1, 0) = w
    _, w, _ = o.lattice(lattice)
    assert np.array_equal(s.get_populations(0)[:, ~fluid], np.repeat(w[:, None], (~fluid).sum(), axis=1))


def test_non_periodic_wall_faces_conserve_mass():
    n = (12, 10, 1)
    N = n[0] * n[1]
    wl = base_wl("D2Q9", n, periodic=(False, False, True), psi_kind=["CS"], eos=[dict(a=1.0, b=4.0, R=1.0, T=0.0802)],
                 G=[[-1.0]])
    rng = np.random.default_rng(8)
    rho0 = 0.15 + 0.05 * rng.uniform(-1, 1, N)
    s = make_oracle(wl, dict(rho=[rho0]))
    m0 = s.get_populations(0).sum()
    s.step(150)
    assert abs(s.get_populations(0).sum() - m0) <= 1e-12 * m0


# ------------------------------------------------------------------ velocity inlet: mass flux rho_w u_w (R10)
@pytest.mark.parametrize("lattice,n", [("D2Q9", (16, 8, 1)), ("D3Q19", (12, 6, 5))])
def test_velocity_inlet_mass_flux(lattice, n):
    """Closed channel (wall at x = nx-1), velocity face at x = 0, y/z periodic:
    every step adds exactly rho_w * u_w per inlet face cell."""
    N = n[0] * n[1] * n[2]
    rho_w, u_w = 0.9, 2e-3
    wl = base_wl(lattice, n, periodic=(False, True, True),
                 face_bc={0: ("VELOCITY", (rho_w,), (u_w, 0, 0))})
    s = make_oracle(wl, dict(rho=[np.ones(N)]))
    m0 = s.get_populations(0).sum()
    steps = 25
    s.step(steps)
    m1 = s.get_populations(0).sum()
    expected = rho_w * u_w * n[1] * n[2] * steps
    assert abs((m1 - m0) - expected) <= 1e-12 * m0


def test_pressure_faces_drive_poiseuille_flow():
    """Pressure (anti-bounce-back) faces at both x ends of a channel with halfway bounce-back walls:
    steady state is Poiseuille flow, u_max = (c_s^2 drho / L) H^2 / (8 nu rho), nu = c_s^2 (tau - 1/2),
    H = ny - 2 (walls half a cell outside the last fluid row), L = nx.  First-order pin of reading R10:
    the O(u^2) terms of the anti-bounce-back formula are NOT pinned by it."""
    nx, ny = 24, 11
    N = nx * ny
    mask = np.zeros((ny, nx), np.uint8)
    mask[0] = mask[-1] = 1
    wl = base_wl("D2Q9", (nx, ny, 1), periodic=(False, True, True),
                 face_bc={0: ("PRESSURE", (1.01,), (0, 0, 0)), 1: ("PRESSURE", (0.99,), (0, 0, 0))})
    s = make_oracle(wl, dict(rho=[np.ones(N)], mask=mask.reshape(-1)))
    s.step(5000)
    rho, u, _ = s.get_macroscopic()
    s.step(200)
    _, u2, _ = s.get_macroscopic()
    assert np.abs(u2 - u).max() < 1e-12          # steady
    ux = u[0].reshape(ny, nx)
    r = rho[0].reshape(ny, nx)
    H, nu = ny - 2, 1.0 / 6.0
    umax = (0.02 / 3.0 / nx) * H * H / (8 * nu)
    assert abs(ux[ny // 2, nx // 2] - umax) < 0.10 * umax
    y = np.arange(ny) - 0.5
    shape = 4 * y * (H - y) / H ** 2
    col = ux[1:-1, nx // 2]
    assert np.abs(col / col.max() - shape[1:-1]).max() < 0.02   # parabolic, zero at the halfway walls
    assert np.all(np.diff(r[ny // 2]) < 0)                      # pressure falls monotonically along x
    assert abs(r[ny // 2, 0] - 1.01) < 2e-3 and abs(r[ny // 2, -1] - 0.99) < 2e-3


# ------------------------------------------------------------------ integer work: link flags and boundary solids
def _brute_link_flags(mask3, e, periodic):
    nz, ny, nx = mask3.shape
    n = (nx, ny, nz)
    flags = np.zeros(mask3.shape, dtype=np.uint32)
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                if mask3[z, y, x]:
                    flags[z, y, x] = 0x80000000
                    continue
                fl = 0
                for i in range(1, len(e)):
                    p = [x - e[i][0], y - e[i][1], z - e[i][2]]
                    out = False
                    for a in range(3):
                        if p[a] < 0 or p[a] >= n[a]:
                            if periodic[a]:
                                p[a] %= n[a]
                            else:
                                out = True
                    if out or mask3[p[2], p[1], p[0]]:
                        fl |= 1 << i
                flags[z, y, x] = fl
    return flags.reshape(-1)


@pytest.mark.parametrize("lattice,n,periodic", [("D2Q9", (9, 7, 1), (True, True, True)),
                                                ("D2Q9", (9, 7, 1), (False, True, True)),
                                                ("D3Q19", (6, 5, 4), (True, False, True))])
def test_link_flags_and_boundary_solids_brute_force(lattice, n, periodic):
    rng = np.random.default_rng(9)
    mask = (rng.uniform(size=n[0] * n[1] * n[2]) < 0.3).astype(np.uint8)
    wl = base_wl(lattice, n, periodic=periodic)
    s = o.Oracle(wl)
    s.set_solid_mask(mask)
    e, _, _ = o.lattice(lattice)
    m3 = mask.reshape(n[2], n[1], n[0])
    assert np.array_equal(s.get_link_flags(), _brute_link_flags(m3, e, periodic))
    # boundary solids: solid with >= 1 fluid neighbour under wrap/clamp indexing
    exp = []
    for idx in range(mask.size):
        if not mask[idx]:
            continue
        x, y, z = idx % n[0], (idx // n[0]) % n[1], idx // (n[0] * n[1])
        hit = False
        for i in range(1, len(e)):
            p = [x + e[i][0], y + e[i][1], z + e[i][2]]
            for a in range(3):
                p[a] = p[a] % n[a] if periodic[a] else min(max(p[a], 0), n[a] - 1)
            if not m3[p[2], p[1], p[0]]:
                hit = True
        if hit:
            exp.append(idx)
    assert np.array_equal(s.get_boundary_solids(), np.array(exp, dtype=np.int64))


# ------------------------------------------------------------------ virtual density (Eq. 17, R11/R12)
def test_virtual_density_uniform_fluid():
    """Next to a uniform fluid of density r the weighted average is r for any neighbourhood shape,
    so rho_s = clamp(phi r - drho, lo, hi) exactly."""
    n = (10, 8, 6)
    N = n[0] * n[1] * n[2]
    rng = np.random.default_rng(10)
    mask = (rng.uniform(size=N) < 0.4).astype(np.uint8)
    wl = base_wl("D3Q19", n, nc=2, wetting=[dict(phi=1.3, drho=0.0, lo=0.0, hi=10.0), dict(phi=1.0, drho=0.25, lo=0.5, hi=10.0)])
    s = make_oracle(wl, dict(rho=[np.full(N, 0.8), np.full(N, 0.6)], mask=mask))
    rho, _, _ = s.get_macroscopic()
    b = s.get_boundary_solids()
    assert np.allclose(rho[0][b], 1.3 * 0.8, rtol=0, atol=1e-15)
    assert np.allclose(rho[1][b], 0.5, rtol=0, atol=1e-15)   # 0.6 - 0.25 = 0.35 -> limiter lo = 0.5
    interior = np.setdiff1d(np.where(mask)[0], b)
    assert np.all(rho[0][interior] == 0)
