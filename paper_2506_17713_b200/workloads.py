"""Seeded synthetic workloads: configuration dicts and input arrays.

This module is the ONE piece shared by the oracle tests and the CUDA path: it
produces plain data (a *workload dict* of parameters plus numpy input arrays)
and holds none of the method's arithmetic (no f_eq, no psi, no force, no EOS).
The oracle (oracle/lbm_oracle.py) and the CUDA binding
(paper_2506_17713_b200/binding.py) each marshal the same dict into their own
configuration struct.

The five configurations are BASELINE.json's ``configs`` (recipes in DESIGN.md
"Input recipe").  Every generator is seeded (numpy PCG64, seed = 1000 + config
number) and takes the domain size as an argument so that the parity tests can
run the same recipe at reduced size.  Physical constants typed here (coexistence
densities, temperatures) are checked against the oracle's Maxwell construction
in tests/test_oracle_eos.py.

Array layout everywhere: flat, x fastest: index = x + nx*(y + ny*z).
"""
from __future__ import annotations

import numpy as np

# --- constants of the configs (verified in tests/test_oracle_eos.py) --------
CS_A, CS_B, CS_R = 1.0, 4.0, 1.0
CS_T_085 = 0.08017625            # 0.85 * T_c, T_c = 0.3773 a/(b R) = 0.094325
CS_RHO_V_085 = 0.0315741         # Maxwell construction at T_r = 0.85
CS_RHO_L_085 = 0.2792816
PR_A, PR_B, PR_R, PR_OMEGA = 2.0 / 49.0, 2.0 / 21.0, 1.0, 0.344
PR_T_07 = 0.05104540285          # 0.7 * T_c, T_c = 0.0778 a/(0.45724 b R)
PR_RHO_V_07 = 0.0556351
PR_RHO_L_07 = 8.0803216

# Wetting parameters of configs 2 and 4 (Eq. 17, second branch): Delta rho of the NON-wetting component at the wall.
# The contact angle has no closed form in (phi, Delta rho): calibrated with the oracle on a flat-walled
# channel (circle fit of the meniscus, tests/test_oracle_physics.py::test_contact_angles_of_configs_2_and_4) --
# 0.32 -> 60 +- 2 deg (config 2), 0.60 -> 40 +- 2 deg (config 4); sweep in DESIGN.md section 4.
C2_DRHO_B = 0.32
C4_DRHO_NW = 0.60

# MRT relaxation rates (reading R9): conserved rows 1.0, s_nu = 1/tau
def mrt_rates(lattice: str, tau: float = 1.0):
    s_nu = 1.0 / tau
    if lattice == "D2Q9":
        # rho, e, eps, jx, qx, jy, qy, pxx, pxy
        return [1.0, 1.19, 1.4, 1.0, 1.2, 1.0, 1.2, s_nu, s_nu]
    # rho, e, eps, jx, qx, jy, qy, jz, qz, 3pxx, 3pixx, pww, piww, pxy, pyz, pxz, mx, my, mz
    return [1.0, 1.19, 1.4, 1.0, 1.2, 1.0, 1.2, 1.0, 1.2, s_nu, 1.4, s_nu, 1.4, s_nu, s_nu, s_nu, 1.98, 1.98, 1.98]


def _rng(config_no: int, extra: int = 0):
    return np.random.Generator(np.random.PCG64(1000 + config_no + 7919 * extra))


def _grid(nx, ny, nz):
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return x.astype(np.float64), y.astype(np.float64), z.astype(np.float64)


def tanh_profile(dist, radius, width, rho_in, rho_out):
    """Eq. 18 of the paper in the corrected form of DESIGN.md reading R14."""
    return 0.5 * (rho_in + rho_out) - 0.5 * (rho_in - rho_out) * np.tanh(2.0 * (dist - radius) / width)


def _min_image(dx, n):
    dx = np.abs(dx)
    return np.minimum(dx, n - dx)


def _round_inputs(arrs, compute_dtype):
    # fp32 runs feed the oracle and the GPU the same fp32-rounded arrays
    if compute_dtype == "f32":
        return [a.astype(np.float32).astype(np.float64) for a in arrs]
    return arrs


# ---------------------------------------------------------------- config 1
def config1(n: int = 64, dtype: str = "f64"):
    """D2Q9 single component, n x n periodic, CS EOS at T_r = 0.85, BGK tau = 1, droplet r = n/4."""
    wl = dict(
        name="C1", lattice="D2Q9", nx=n, ny=n, nz=1, n_components=1, periodic=(True, True, True),
        psi_kind=["CS"], eos=[dict(a=CS_A, b=CS_B, R=CS_R, T=CS_T_085, alpha=1.0)], G=[[-1.0]],
        collision="BGK", tau=[1.0], forcing="EDM", compute_dtype=dtype, store_dtype=dtype, steps=2000,
    )
    x, y, _ = _grid(n, n, 1)
    c = (n - 1) / 2.0
    dist = np.sqrt((x - c) ** 2 + (y - c) ** 2)
    rho = tanh_profile(dist, n / 4.0, 2.0, CS_RHO_L_085, CS_RHO_V_085)
    rho = rho + _rng(1).uniform(-1e-3, 1e-3, size=rho.shape)
    (rho,) = _round_inputs([rho.reshape(-1)], dtype)
    return wl, dict(rho=[rho], u=None, mask=None)


# ---------------------------------------------------------------- config 2
def config2(nx: int = 512, ny: int = 256, dtype: str = "f32", wall: int = 8, drho_b: float = C2_DRHO_B):
    """D2Q9 two components between two solid plates (capillary geometry), SC93 psi, G_AB = 3.5 classic."""
    g_ab = 3.5 / 3.0  # classic SC93 G = 3.5 with weights w_i  ==  g = 3.5*c_s^2 with weights w_i/c_s^2 (R15)
    wl = dict(
        name="C2", lattice="D2Q9", nx=nx, ny=ny, nz=1, n_components=2, periodic=(True, True, True),
        psi_kind=["SC93", "SC93"], eos=[dict(rho0=1.0), dict(rho0=1.0)],
        G=[[0.0, g_ab], [g_ab, 0.0]],
        wetting=[dict(phi=1.0, drho=0.0, lo=0.0, hi=1.2), dict(phi=1.0, drho=drho_b, lo=0.0, hi=1.2)],
        collision="BGK", tau=[1.0, 1.0], forcing="EDM", compute_dtype=dtype, store_dtype=dtype, steps=20000,
    )
    x, y, _ = _grid(nx, ny, 1)
    mask = ((y < wall) | (y >= ny - wall)).astype(np.uint8)
    a = np.where(x < nx // 4, 1.0, 0.03)
    b = np.where(x < nx // 4, 0.03, 1.0)
    r = _rng(2)
    a = a + r.uniform(-1e-3, 1e-3, size=a.shape)
    b = b + r.uniform(-1e-3, 1e-3, size=b.shape)
    a, b = _round_inputs([a.reshape(-1), b.reshape(-1)], dtype)
    return wl, dict(rho=[a, b], u=None, mask=mask.reshape(-1))


# ---------------------------------------------------------------- config 3
def config3(n: int = 256, dtype: str = "f32", alpha: float = 0.5):
    """D3Q19 single component, n^3 periodic, PR EOS at T_r = 0.7, MRT, EDM; spinodal decomposition."""
    wl = dict(
        name="C3", lattice="D3Q19", nx=n, ny=n, nz=n, n_components=1, periodic=(True, True, True),
        psi_kind=["PR"], eos=[dict(a=PR_A, b=PR_B, R=PR_R, omega=PR_OMEGA, T=PR_T_07, alpha=alpha)], G=[[-1.0]],
        collision="MRT", tau=[1.0], mrt_rates=[mrt_rates("D3Q19", 1.0)], forcing="EDM",
        compute_dtype=dtype, store_dtype=dtype, steps=1000,
    )
    mean = 0.5 * (PR_RHO_L_07 + PR_RHO_V_07)
    rho = mean + _rng(3).normal(0.0, 1e-2, size=n * n * n)
    (rho,) = _round_inputs([rho], dtype)
    return wl, dict(rho=[rho], u=None, mask=None)


# ---------------------------------------------------------------- config 4
def sphere_pack_mask(nx, ny, nz, porosity=0.20, rmin=6.0, rmax=14.0, buffer=8, seed_no=4):
    """Seeded overlapping-sphere solid mask, periodic in y and z, solid-free buffers at both x ends;
    pore cells not 6-connected (periodically in y, z) to the inlet plane are filled.
    Returns (mask uint8 [N], porosity of the core x in [buffer, nx-buffer))."""
    from scipy import ndimage
    from scipy.sparse import coo_matrix
    from scipy.sparse.csgraph import connected_components

    r = _rng(seed_no, 1)
    solid = np.zeros((nz, ny, nx), dtype=bool)
    core = slice(buffer, nx - buffer)
    ncore = (nx - 2 * buffer) * ny * nz
    # radii scale with the box so that reduced-size tests keep several spheres
    scale = min(1.0, min(nx, ny, nz) / 100.0)
    rmin, rmax = max(2.0, rmin * scale), max(3.0, rmax * scale)
    npore = ncore          # pore cells of the core, tracked incrementally
    guard = 0
    while npore / ncore > porosity and guard < 2000000:
        guard += 1
        cx, cy, cz = r.uniform(0, nx), r.uniform(0, ny), r.uniform(0, nz)
        rad = r.uniform(rmin, rmax)
        x0, x1 = int(max(buffer, np.floor(cx - rad))), int(min(nx - buffer, np.ceil(cx + rad) + 1))
        if x0 >= x1:
            continue
        ys = np.arange(int(np.floor(cy - rad)), int(np.ceil(cy + rad)) + 1)
        zs = np.arange(int(np.floor(cz - rad)), int(np.ceil(cz + rad)) + 1)
        if len(ys) >= ny or len(zs) >= nz:   # tiny test boxes: a sphere may not wrap onto itself
            continue
        xs = np.arange(x0, x1)
        d2 = ((zs[:, None, None] - cz) ** 2 + (ys[None, :, None] - cy) ** 2 + (xs[None, None, :] - cx) ** 2)
        ball = d2 <= rad * rad
        ix = np.ix_(zs % nz, ys % ny, xs)
        sub = solid[ix]
        npore -= int((ball & ~sub).sum())
        solid[ix] = sub | ball
    # keep only the pore space connected to the inlet plane: label without wrap, then join labels that
    # touch across the periodic y and z faces, and keep the groups that reach x = 0
    pore = ~solid
    lab, nlab = ndimage.label(pore)
    pairs = []
    for a_, b_ in ((lab[0, :, :], lab[-1, :, :]), (lab[:, 0, :], lab[:, -1, :])):
        both = (a_ > 0) & (b_ > 0)
        if both.any():
            pairs.append(np.unique(np.stack([a_[both], b_[both]], axis=1), axis=0))
    if pairs:
        pr = np.concatenate(pairs, axis=0)
        g = coo_matrix((np.ones(len(pr), dtype=np.int8), (pr[:, 0], pr[:, 1])), shape=(nlab + 1, nlab + 1))
        _, group = connected_components(g, directed=False)
    else:
        group = np.arange(nlab + 1)
    inlet = np.unique(lab[:, :, 0])
    inlet = inlet[inlet > 0]
    keep_group = np.zeros(group.max() + 1, dtype=bool)
    keep_group[group[inlet]] = True
    keep_label = keep_group[group]
    keep_label[0] = False
    solid = ~keep_label[lab]
    por = float((~solid[:, :, core]).sum() / ncore)
    return solid.astype(np.uint8).reshape(-1), por


def config4(n: int = 400, store_dtype: str = "f16", drho_nw: float = C4_DRHO_NW, buffer: int = 8):
    """D3Q19 two components in a seeded sphere pack; velocity inlet x=0 (non-wetting), pressure outlet x=n-1."""
    g_ab = 3.5 / 3.0
    buffer = min(buffer, max(2, n // 8))
    wl = dict(
        name="C4", lattice="D3Q19", nx=n, ny=n, nz=n, n_components=2, periodic=(False, True, True),
        psi_kind=["SC93", "SC93"], eos=[dict(rho0=1.0), dict(rho0=1.0)],
        G=[[0.0, g_ab], [g_ab, 0.0]],
        # component 0 = non-wetting (injected), component 1 = wetting
        wetting=[dict(phi=1.0, drho=drho_nw, lo=0.0, hi=1.2), dict(phi=1.0, drho=0.0, lo=0.0, hi=1.2)],
        collision="BGK", tau=[1.0, 1.0], forcing="EDM", compute_dtype="f32", store_dtype=store_dtype, steps=5000,
        face_bc={0: ("VELOCITY", (1.0, 0.03), (1e-3, 0.0, 0.0)), 1: ("PRESSURE", (0.03, 1.0), (0.0, 0.0, 0.0))},
    )
    mask, por = sphere_pack_mask(n, n, n, porosity=0.20, buffer=buffer)
    wl["porosity"] = por                                  # of the core x in [buffer, n-buffer)
    wl["fluid_fraction"] = float(1.0 - mask.mean())       # of the whole box
    x, _, _ = _grid(n, n, n)
    nw = np.where(x < buffer, 1.0, 0.03)
    w = np.where(x < buffer, 0.03, 1.0)
    nw, w = _round_inputs([nw.reshape(-1), w.reshape(-1)], "f32")
    return wl, dict(rho=[nw, w], u=None, mask=mask)


# ---------------------------------------------------------------- config 5
def config5(n: int = 512, dtype: str = "f32", store_dtype: str | None = None):
    """D3Q19 single component CS multiphase, n^3 periodic, BGK; seeded droplets in vapour."""
    wl = dict(
        name="C5", lattice="D3Q19", nx=n, ny=n, nz=n, n_components=1, periodic=(True, True, True),
        psi_kind=["CS"], eos=[dict(a=CS_A, b=CS_B, R=CS_R, T=CS_T_085, alpha=1.0)], G=[[-1.0]],
        collision="BGK", tau=[1.0], forcing="EDM", compute_dtype=dtype, store_dtype=store_dtype or dtype, steps=500,
    )
    ndrop = max(1, int(round(64 * (n / 512.0) ** 3)))
    r = _rng(5)
    # radii U[10,30] at full size; shrunk with the box below 128 so reduced tests still hold droplets
    s = min(1.0, n / 128.0)
    cen = r.uniform(0, n, size=(ndrop, 3))
    rad = r.uniform(10.0 * s, 30.0 * s, size=ndrop)
    rho = np.full((n, n, n), CS_RHO_V_085, dtype=np.float64)
    ax = np.arange(n, dtype=np.float64)
    for (cx, cy, cz), rr in zip(cen, rad):
        dx2 = _min_image(ax - cx, n) ** 2
        dy2 = _min_image(ax - cy, n) ** 2
        dz2 = _min_image(ax - cz, n) ** 2
        # only touch the bounding box of the droplet (+ interface) to keep 512^3 generation fast
        reach = rr + 8.0
        zi = np.where(dz2 <= reach * reach)[0]
        yi = np.where(dy2 <= reach * reach)[0]
        xi = np.where(dx2 <= reach * reach)[0]
        dist = np.sqrt(dz2[zi][:, None, None] + dy2[yi][None, :, None] + dx2[xi][None, None, :])
        prof = tanh_profile(dist, rr, 2.0, CS_RHO_L_085, CS_RHO_V_085)
        sub = rho[np.ix_(zi, yi, xi)]
        rho[np.ix_(zi, yi, xi)] = np.maximum(sub, prof)
    (rho,) = _round_inputs([rho.reshape(-1)], dtype)
    return wl, dict(rho=[rho], u=None, mask=None)


# ---------------------------------------------------------------- paper §4 workload (NEXT-4)
def paper_benchmark(n: int = 416, dtype: str = "f32", store_dtype: str | None = None):
    """The paper's own performance case: D3Q19, BGK, droplet R=30 in vapour,
    psi = exp(-1/rho), fully periodic.  g = -10/3 gives rho_l/rho_v ~ 7.6."""
    wl = dict(
        name="P4", lattice="D3Q19", nx=n, ny=n, nz=n, n_components=1, periodic=(True, True, True),
        psi_kind=["EXP"], eos=[dict()], G=[[-10.0 / 3.0]],
        collision="BGK", tau=[1.0], forcing="EDM", compute_dtype=dtype, store_dtype=store_dtype or dtype, steps=500,
    )
    ax = np.arange(n, dtype=np.float64) - (n - 1) / 2.0
    dist = np.sqrt(ax[:, None, None] ** 2 + ax[None, :, None] ** 2 + ax[None, None, :] ** 2)
    rr = 30.0 * min(1.0, n / 128.0)
    rho = tanh_profile(dist, rr, 3.0, 2.7828, 0.3675)
    (rho,) = _round_inputs([rho.reshape(-1)], dtype)
    return wl, dict(rho=[rho], u=None, mask=None)


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}
