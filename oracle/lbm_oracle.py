"""ctypes wrapper around oracle/lbm_oracle.cpp.

ORACLE — TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
imports nothing from paper_2506_17713_b200 and shares no code with the CUDA path.

The neutral *workload dict* (plain data, produced by
paper_2506_17713_b200.workloads) is marshalled here into the oracle's own
``olbm_config`` struct; the CUDA binding marshals the same dict into its own
``lbm_config_t``.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "lbm_oracle.cpp"
_LIB = _HERE / "liblbm_oracle.so"

LATTICES = {"D2Q9": 0, "D3Q19": 1}
PSI_KINDS = {"CS": 0, "PR": 1, "VDW": 2, "RK": 3, "RKS": 4, "RHO": 5, "EXP": 6, "SC93": 7}
COLLISIONS = {"BGK": 0, "MRT": 1}
FORCINGS = {"EDM": 0, "SHIFT": 1}
DTYPES = {"f16": 0, "f32": 1, "f64": 2}
FACE_KINDS = {"PERIODIC": 0, "WALL": 1, "VELOCITY": 2, "PRESSURE": 3}


class _Config(C.Structure):
    _fields_ = [
        ("lattice", C.c_int32),
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("n_components", C.c_int32),
        ("periodic", C.c_int32 * 3),
        ("psi_kind", C.c_int32 * 2),
        ("collision", C.c_int32),
        ("forcing", C.c_int32),
        ("compute_dtype", C.c_int32),
        ("store_dtype", C.c_int32),
        ("no_collide", C.c_int32),
        ("eos_a", C.c_double * 2), ("eos_b", C.c_double * 2), ("eos_R", C.c_double * 2),
        ("eos_omega", C.c_double * 2), ("eos_T", C.c_double * 2),
        ("alpha", C.c_double * 2),
        ("rho0", C.c_double * 2),
        ("G", (C.c_double * 2) * 2),
        ("wet_phi", C.c_double * 2), ("wet_drho", C.c_double * 2),
        ("wet_lo", C.c_double * 2), ("wet_hi", C.c_double * 2),
        ("tau", C.c_double * 2),
        ("mrt_rates", (C.c_double * 19) * 2),
        ("rho_ref", C.c_double),
        ("zc_A", C.c_double * 2),
        ("body_accel", C.c_double * 3),
        ("st_kappa", C.c_double * 2),
    ]


def build(force: bool = False) -> Path:
    """Compile the oracle with g++ (-O2, no FMA contraction, OpenMP over the outer loops)."""
    if _LIB.exists() and not force and _LIB.stat().st_mtime >= _SRC.stat().st_mtime:
        return _LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           str(_SRC), "-o", str(_LIB)]
    subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        L.olbm_create.restype = C.c_void_p
        L.olbm_create.argtypes = [C.POINTER(_Config)]
        L.olbm_destroy.argtypes = [C.c_void_p]
        L.olbm_destroy.restype = None
        L.olbm_set_solid_mask.argtypes = [C.c_void_p, C.c_void_p]
        L.olbm_set_face_bc.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.olbm_init_fields.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.olbm_step.argtypes = [C.c_void_p, C.c_int]
        L.olbm_get_macroscopic.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.olbm_get_populations.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.olbm_set_populations.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.olbm_get_link_flags.argtypes = [C.c_void_p, C.c_void_p]
        L.olbm_get_boundary_solids.argtypes = [C.c_void_p, C.c_void_p, C.c_int64]
        L.olbm_get_boundary_solids.restype = C.c_int64
        L.olbm_get_force.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.olbm_get_psi.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.olbm_lattice.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.olbm_feq.argtypes = [C.c_int, C.c_double, C.c_void_p, C.c_void_p]
        L.olbm_mrt_matrices.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
        L.olbm_eos_critical_temperature.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double]
        L.olbm_eos_critical_temperature.restype = C.c_double
        L.olbm_eos_pressure.argtypes = [C.c_int] + [C.c_double] * 5 + [C.c_void_p, C.c_void_p, C.c_int64]
        L.olbm_round_to_half.argtypes = [C.c_float]
        L.olbm_round_to_half.restype = C.c_float
        L.olbm_set_threads.argtypes = [C.c_int]
        L.olbm_config_size.restype = C.c_int
        assert L.olbm_config_size() == C.sizeof(_Config), "olbm_config layout mismatch"
        _lib = L
    return _lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def make_config(wl: dict) -> _Config:
    """Marshal the neutral workload dict into olbm_config."""
    c = _Config()
    c.lattice = LATTICES[wl["lattice"]]
    c.nx, c.ny, c.nz = int(wl["nx"]), int(wl["ny"]), int(wl.get("nz", 1))
    nc = int(wl.get("n_components", 1))
    c.n_components = nc
    per = wl.get("periodic", (True, True, True))
    for a in range(3):
        c.periodic[a] = 1 if per[a] else 0
    c.collision = COLLISIONS[wl.get("collision", "BGK")]
    c.forcing = FORCINGS[wl.get("forcing", "EDM")]
    c.compute_dtype = DTYPES[wl.get("compute_dtype", "f64")]
    c.store_dtype = DTYPES[wl.get("store_dtype", wl.get("compute_dtype", "f64"))]
    c.no_collide = 1 if wl.get("no_collide", False) else 0
    c.rho_ref = float(wl.get("rho_ref", 0.0))
    q = 9 if wl["lattice"] == "D2Q9" else 19
    G = wl.get("G", [[0.0] * nc for _ in range(nc)])
    for k in range(nc):
        c.psi_kind[k] = PSI_KINDS[wl["psi_kind"][k]]
        eos = wl.get("eos", [{}] * nc)[k]
        c.eos_a[k] = float(eos.get("a", 0.0))
        c.eos_b[k] = float(eos.get("b", 0.0))
        c.eos_R[k] = float(eos.get("R", 1.0))
        c.eos_omega[k] = float(eos.get("omega", 0.0))
        c.eos_T[k] = float(eos.get("T", 0.0))
        c.alpha[k] = float(eos.get("alpha", 1.0))
        c.rho0[k] = float(eos.get("rho0", 1.0))
        wet = wl.get("wetting", [{}] * nc)[k]
        c.wet_phi[k] = float(wet.get("phi", 1.0))
        c.wet_drho[k] = float(wet.get("drho", 0.0))
        c.wet_lo[k] = float(wet.get("lo", 0.0))
        c.wet_hi[k] = float(wet.get("hi", 1e30))
        c.tau[k] = float(wl.get("tau", [1.0] * nc)[k])
        rates = wl.get("mrt_rates")
        for r in range(q):
            c.mrt_rates[k][r] = float(rates[k][r]) if rates is not None else 1.0 / c.tau[k]
        for kp in range(nc):
            c.G[k][kp] = float(G[k][kp])
        c.zc_A[k] = float(wl.get("zc_A", [0.0] * nc)[k])
    for a in range(3):
        c.body_accel[a] = float(wl.get("body_accel", (0.0, 0.0, 0.0))[a])
    for k in range(nc):
        c.st_kappa[k] = float(wl.get("st_kappa", [0.0] * nc)[k])
    return c


class Oracle:
    """One oracle simulation.  Arrays are flat, x fastest: index = x + nx*(y + ny*z)."""

    def __init__(self, wl: dict):
        self.wl = wl
        self.cfg = make_config(wl)
        self.L = lib()
        self.h = self.L.olbm_create(C.byref(self.cfg))
        if not self.h:
            raise ValueError("oracle rejected the configuration")
        self.nc = self.cfg.n_components
        self.q = 9 if self.cfg.lattice == 0 else 19
        self.d = 2 if self.cfg.lattice == 0 else 3
        self.N = self.cfg.nx * self.cfg.ny * self.cfg.nz
        for face, (kind, rho_w, u_w) in wl.get("face_bc", {}).items():
            self.set_face_bc(int(face), kind, rho_w, u_w)

    def __del__(self):
        if getattr(self, "h", None):
            self.L.olbm_destroy(self.h)
            self.h = None

    def set_solid_mask(self, mask: np.ndarray):
        m = np.ascontiguousarray(mask, dtype=np.uint8).reshape(-1)
        assert m.size == self.N
        assert self.L.olbm_set_solid_mask(self.h, _ptr(m)) == 0

    def set_face_bc(self, face: int, kind: str, rho_w, u_w):
        r = np.zeros(2, dtype=np.float64)
        r[: len(rho_w)] = rho_w
        u = np.zeros(3, dtype=np.float64)
        u[: len(u_w)] = u_w
        rc = self.L.olbm_set_face_bc(self.h, face, FACE_KINDS[kind], _ptr(r), _ptr(u))
        if rc != 0:
            raise ValueError("invalid face boundary condition")

    def init_fields(self, rho, u=None):
        rho = [np.ascontiguousarray(r, dtype=np.float64).reshape(-1) for r in rho]
        assert len(rho) == self.nc and all(r.size == self.N for r in rho)
        ptrs = (C.c_void_p * self.nc)(*[r.ctypes.data for r in rho])
        up = None
        if u is not None:
            u = np.ascontiguousarray(u, dtype=np.float64).reshape(-1)
            assert u.size == self.d * self.N
            up = _ptr(u)
        assert self.L.olbm_init_fields(self.h, ptrs, up) == 0

    def step(self, n: int = 1):
        assert self.L.olbm_step(self.h, int(n)) == 0

    def get_macroscopic(self):
        rho = [np.empty(self.N, dtype=np.float64) for _ in range(self.nc)]
        u = np.empty((self.d, self.N), dtype=np.float64)
        p = np.empty(self.N, dtype=np.float64)
        ptrs = (C.c_void_p * self.nc)(*[r.ctypes.data for r in rho])
        assert self.L.olbm_get_macroscopic(self.h, ptrs, _ptr(u), _ptr(p)) == 0
        return rho, u, p

    def get_populations(self, k: int = 0) -> np.ndarray:
        out = np.empty((self.q, self.N), dtype=np.float64)
        assert self.L.olbm_get_populations(self.h, k, _ptr(out)) == 0
        return out

    def set_populations(self, k: int, f: np.ndarray):
        f = np.ascontiguousarray(f, dtype=np.float64)
        assert f.shape == (self.q, self.N)
        assert self.L.olbm_set_populations(self.h, k, _ptr(f)) == 0

    def get_link_flags(self) -> np.ndarray:
        out = np.empty(self.N, dtype=np.uint32)
        assert self.L.olbm_get_link_flags(self.h, _ptr(out)) == 0
        return out

    def get_boundary_solids(self) -> np.ndarray:
        m = self.L.olbm_get_boundary_solids(self.h, None, 0)
        out = np.empty(m, dtype=np.int64)
        if m:
            self.L.olbm_get_boundary_solids(self.h, _ptr(out), m)
        return out

    def get_force(self, k: int = 0) -> np.ndarray:
        out = np.empty((self.d, self.N), dtype=np.float64)
        assert self.L.olbm_get_force(self.h, k, _ptr(out)) == 0
        return out

    def get_psi(self, k: int = 0) -> np.ndarray:
        out = np.empty(self.N, dtype=np.float64)
        assert self.L.olbm_get_psi(self.h, k, _ptr(out)) == 0
        return out


# ---- stand-alone pieces ---------------------------------------------------
def lattice(name: str):
    q = C.c_int(0)
    e = np.zeros((19, 3), dtype=np.int32)
    w = np.zeros(19, dtype=np.float64)
    opp = np.zeros(19, dtype=np.int32)
    lib().olbm_lattice(LATTICES[name], C.byref(q), _ptr(e), _ptr(w), _ptr(opp))
    return e[: q.value].copy(), w[: q.value].copy(), opp[: q.value].copy()


def feq(name: str, rho: float, u) -> np.ndarray:
    uu = np.zeros(3, dtype=np.float64)
    uu[: len(u)] = u
    out = np.zeros(19, dtype=np.float64)
    q = lib().olbm_feq(LATTICES[name], float(rho), _ptr(uu), _ptr(out))
    return out[:q].copy()


def mrt_matrices(name: str):
    q = 9 if name == "D2Q9" else 19
    M = np.zeros((q, q), dtype=np.float64)
    Mi = np.zeros((q, q), dtype=np.float64)
    lib().olbm_mrt_matrices(LATTICES[name], _ptr(M), _ptr(Mi))
    return M, Mi


def eos_critical_temperature(kind: str, a: float, b: float, R: float = 1.0) -> float:
    return lib().olbm_eos_critical_temperature(PSI_KINDS[kind], a, b, R)


def eos_pressure(kind: str, a, b, R, omega, T, rho) -> np.ndarray:
    rho = np.ascontiguousarray(np.atleast_1d(rho), dtype=np.float64)
    p = np.empty_like(rho)
    lib().olbm_eos_pressure(PSI_KINDS[kind], a, b, R, omega, T, _ptr(rho), _ptr(p), rho.size)
    return p


def round_to_half(v: float) -> float:
    return float(lib().olbm_round_to_half(C.c_float(v)))


def set_threads(n: int) -> int:
    return int(lib().olbm_set_threads(int(n)))


def host_cores() -> int:
    return os.cpu_count() or 1
