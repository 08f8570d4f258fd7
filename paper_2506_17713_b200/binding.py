"""Thin Python binding of the C-ABI in include/lbm.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of liblbm_b200.so; PyTorch is used here only
to allocate the device workspace and to name the CUDA stream.  There is no CPU fallback: if the
library has not been built (``python paper_2506_17713_b200/build.py`` or
``__graft_entry__.build()``) importing the symbols raises.

The module exposes the raw C functions under their C names (``lbm_create``, ``lbm_step``, ...)
and a small convenience class ``LBM`` that owns a workspace tensor and a handle.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "liblbm_b200.so"

LBM_OK = 0
LATTICES = {"D2Q9": 0, "D3Q19": 1}
PSI_KINDS = {"CS": 0, "PR": 1, "VDW": 2, "RK": 3, "RKS": 4, "RHO": 5, "EXP": 6, "SC93": 7}
COLLISIONS = {"BGK": 0, "MRT": 1}
FORCINGS = {"EDM": 0, "SHIFT": 1}
DTYPES = {"f16": 0, "f32": 1, "f64": 2}
FACE_KINDS = {"PERIODIC": 0, "WALL": 1, "VELOCITY": 2, "PRESSURE": 3}
KERNEL_IDS = {"moments": 0, "virtual": 1, "step": 2, "fused": 3, "persistent": 4}
FLAG_NO_COLLIDE = 1
FLAG_TWO_PASS = 2
FLAG_ONE_PASS = 4
STATUS = {0: "LBM_OK", -1: "LBM_E_INVALID", -2: "LBM_E_UNSUPPORTED", -3: "LBM_E_NOMEM", -4: "LBM_E_CUDA",
          -5: "LBM_E_STATE"}


class lbm_eos_t(C.Structure):
    _fields_ = [("psi_kind", C.c_int32), ("pad_", C.c_int32), ("a", C.c_double), ("b", C.c_double), ("R", C.c_double),
                ("omega", C.c_double), ("T", C.c_double), ("alpha", C.c_double), ("rho0", C.c_double)]


class lbm_wetting_t(C.Structure):
    _fields_ = [("phi", C.c_double), ("drho", C.c_double), ("lo", C.c_double), ("hi", C.c_double)]


class lbm_config_t(C.Structure):
    _fields_ = [
        ("lattice", C.c_int32), ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("n_components", C.c_int32), ("periodic", C.c_int32 * 3),
        ("collision", C.c_int32), ("forcing", C.c_int32), ("compute_dtype", C.c_int32), ("store_dtype", C.c_int32),
        ("flags", C.c_uint32), ("pad_", C.c_int32),
        ("eos", lbm_eos_t * 2), ("G", (C.c_double * 2) * 2), ("wet", lbm_wetting_t * 2),
        ("tau", C.c_double * 2), ("mrt_rates", (C.c_double * 19) * 2), ("rho_ref", C.c_double), ("zc_A", C.c_double * 2), ("body_accel", C.c_double * 3), ("st_kappa", C.c_double * 2),
    ]


class LBMError(RuntimeError):
    pass


_lib = None

_SIGNATURES = {
    "lbm_workspace_bytes": (C.c_size_t, [C.POINTER(lbm_config_t)]),
    "lbm_create": (C.c_int, [C.POINTER(lbm_config_t), C.c_void_p, C.c_size_t, C.c_void_p, C.POINTER(C.c_void_p)]),
    "lbm_destroy": (None, [C.c_void_p]),
    "lbm_set_solid_mask": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int]),
    "lbm_set_face_bc": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]),
    "lbm_init_fields": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int]),
    "lbm_step": (C.c_int, [C.c_void_p, C.c_int]),
    "lbm_get_macroscopic": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int]),
    "lbm_get_populations": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_int]),
    "lbm_set_populations": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_int]),
    "lbm_get_link_flags": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int]),
    "lbm_get_boundary_solids": (C.c_int64, [C.c_void_p, C.c_void_p, C.c_int64]),
    "lbm_get_psi": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_int]),
    "lbm_render_isosurface": (C.c_int, [C.c_void_p, C.c_int, C.c_double, C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_int]),
    "lbm_get_lattice": (C.c_int, [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "lbm_set_profiling": (C.c_int, [C.c_void_p, C.c_int]),
    "lbm_get_kernel_times": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "lbm_halo_bytes": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p]),
    "lbm_export_halo": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_void_p]),
    "lbm_import_halo": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_void_p]),
    "lbm_step_noalloc": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "lbm_noalloc_max_scratch_bytes": (C.c_size_t, []),
    "lbm_noalloc_last_error": (C.c_char_p, []),
    "lbm_hot_path": (C.c_int, [C.c_void_p]),
    "lbm_steps_done": (C.c_int64, [C.c_void_p]),
    "lbm_kernel_launches": (C.c_int64, [C.c_void_p]),
    "lbm_last_error": (C.c_char_p, [C.c_void_p]),
    "lbm_version": (C.c_char_p, []),
    "lbm_config_bytes": (C.c_size_t, []),
}


def load_library():
    """dlopen liblbm_b200.so and declare the prototypes.  Raises if the library is missing."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise LBMError(f"CUDA extension missing: {LIB_PATH} (run paper_2506_17713_b200/build.py); "
                           "there is no CPU fallback")
        L = C.CDLL(str(LIB_PATH))
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        if L.lbm_config_bytes() != C.sizeof(lbm_config_t):
            raise LBMError("lbm_config_t layout mismatch between binding.py and liblbm_b200.so")
        _lib = L
    return _lib


def __getattr__(name):  # lbm_create, lbm_step, ... as module attributes
    if name in _SIGNATURES:
        return getattr(load_library(), name)
    raise AttributeError(name)


def make_config(wl: dict) -> lbm_config_t:
    """Marshal the neutral workload dict (paper_2506_17713_b200.workloads) into lbm_config_t."""
    c = lbm_config_t()
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
    c.flags = FLAG_NO_COLLIDE if wl.get("no_collide", False) else 0
    c.flags |= {None: 0, "two_pass": FLAG_TWO_PASS, "one_pass": FLAG_ONE_PASS}[wl.get("path")]
    c.rho_ref = float(wl.get("rho_ref", 0.0))
    q = 9 if wl["lattice"] == "D2Q9" else 19
    G = wl.get("G", [[0.0] * nc for _ in range(nc)])
    for k in range(nc):
        eos = wl.get("eos", [{}] * nc)[k]
        c.eos[k].psi_kind = PSI_KINDS[wl["psi_kind"][k]]
        c.eos[k].a = float(eos.get("a", 0.0))
        c.eos[k].b = float(eos.get("b", 0.0))
        c.eos[k].R = float(eos.get("R", 1.0))
        c.eos[k].omega = float(eos.get("omega", 0.0))
        c.eos[k].T = float(eos.get("T", 0.0))
        c.eos[k].alpha = float(eos.get("alpha", 1.0))
        c.eos[k].rho0 = float(eos.get("rho0", 1.0))
        wet = wl.get("wetting", [{}] * nc)[k]
        c.wet[k].phi = float(wet.get("phi", 1.0))
        c.wet[k].drho = float(wet.get("drho", 0.0))
        c.wet[k].lo = float(wet.get("lo", 0.0))
        c.wet[k].hi = float(wet.get("hi", 1e30))
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


def _np_dtype_code(a: np.ndarray) -> int:
    if a.dtype == np.float32:
        return DTYPES["f32"]
    if a.dtype == np.float64:
        return DTYPES["f64"]
    raise TypeError("arrays must be float32 or float64")


class LBM:
    """One simulation on one GPU.  Owns the device workspace (a torch uint8 tensor) and the handle."""

    def __init__(self, wl: dict, device: str = "cuda:0", stream=None):
        import torch

        self.L = load_library()
        if not torch.cuda.is_available():
            raise LBMError("no CUDA device: the Shan-Chen LBM path has no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        self.wl = wl
        self.cfg = make_config(wl)
        nbytes = self.L.lbm_workspace_bytes(C.byref(self.cfg))
        if nbytes == 0:
            raise LBMError("invalid configuration")
        self.nc = self.cfg.n_components
        self.q = 9 if self.cfg.lattice == 0 else 19
        self.d = 2 if self.cfg.lattice == 0 else 3
        self.N = self.cfg.nx * self.cfg.ny * self.cfg.nz
        self.workspace_bytes = nbytes
        with torch.cuda.device(self.device):
            self.ws = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            rc = self.L.lbm_create(C.byref(self.cfg), C.c_void_p(self.ws.data_ptr()), nbytes,
                                   C.c_void_p(self.stream.cuda_stream), C.byref(h))
        if rc != LBM_OK:
            raise LBMError(f"lbm_create failed: {STATUS.get(rc, rc)}")
        self.h = h
        for face, (kind, rho_w, u_w) in wl.get("face_bc", {}).items():
            self.set_face_bc(int(face), kind, rho_w, u_w)

    # -- helpers -----------------------------------------------------------
    def _check(self, rc, what):
        if rc != LBM_OK:
            msg = self.L.lbm_last_error(self.h)
            raise LBMError(f"{what} failed: {STATUS.get(rc, rc)}: {msg.decode() if msg else ''}")

    def close(self):
        if getattr(self, "h", None):
            self.torch.cuda.synchronize(self.device)
            self.L.lbm_destroy(self.h)
            self.h = None
            self.ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ct_torch(self):
        return self.torch.float32 if self.cfg.compute_dtype == DTYPES["f32"] else self.torch.float64

    # -- C-ABI calls ---------------------------------------------------------
    def set_solid_mask(self, mask):
        if isinstance(mask, np.ndarray):
            m = np.ascontiguousarray(mask, dtype=np.uint8).reshape(-1)
            assert m.size == self.N
            self._check(self.L.lbm_set_solid_mask(self.h, m.ctypes.data_as(C.c_void_p), 0), "lbm_set_solid_mask")
        else:  # torch uint8 tensor on the device
            assert mask.numel() == self.N and mask.dtype == self.torch.uint8 and mask.is_cuda
            self._check(self.L.lbm_set_solid_mask(self.h, C.c_void_p(mask.data_ptr()), 1), "lbm_set_solid_mask")

    def set_face_bc(self, face: int, kind: str, rho_w, u_w):
        r = np.zeros(2, dtype=np.float64)
        r[: len(rho_w)] = rho_w
        u = np.zeros(3, dtype=np.float64)
        u[: len(u_w)] = u_w
        self._check(self.L.lbm_set_face_bc(self.h, face, FACE_KINDS[kind], r.ctypes.data_as(C.c_void_p),
                                           u.ctypes.data_as(C.c_void_p)), "lbm_set_face_bc")

    def init_fields(self, rho, u=None):
        """rho: list of n_components arrays (numpy float32/float64 on the host, or torch CUDA tensors)."""
        assert len(rho) == self.nc
        if isinstance(rho[0], np.ndarray):
            arrs = [np.ascontiguousarray(r).reshape(-1) for r in rho]
            code = _np_dtype_code(arrs[0])
            assert all(a.size == self.N and _np_dtype_code(a) == code for a in arrs)
            ptrs = (C.c_void_p * self.nc)(*[a.ctypes.data for a in arrs])
            up = None
            if u is not None:
                uu = np.ascontiguousarray(u, dtype=arrs[0].dtype).reshape(-1)
                assert uu.size == self.d * self.N
                up = uu.ctypes.data_as(C.c_void_p)
            self._check(self.L.lbm_init_fields(self.h, ptrs, up, code, 0), "lbm_init_fields")
        else:
            t = self.torch
            arrs = [r.contiguous().view(-1) for r in rho]
            code = DTYPES["f32"] if arrs[0].dtype == t.float32 else DTYPES["f64"]
            assert all(a.numel() == self.N and a.is_cuda and a.dtype == arrs[0].dtype for a in arrs)
            ptrs = (C.c_void_p * self.nc)(*[a.data_ptr() for a in arrs])
            up = None
            if u is not None:
                uu = u.contiguous().view(-1)
                assert uu.numel() == self.d * self.N and uu.dtype == arrs[0].dtype
                up = C.c_void_p(uu.data_ptr())
            self._check(self.L.lbm_init_fields(self.h, ptrs, up, code, 1), "lbm_init_fields")

    def step(self, n: int = 1):
        self._check(self.L.lbm_step(self.h, int(n)), "lbm_step")

    def get_macroscopic(self, dtype=np.float64, want_u=True, want_p=True):
        """Host copies (numpy): rho list, u [d,N], p [N]."""
        code = DTYPES["f32"] if dtype == np.float32 else DTYPES["f64"]
        rho = [np.empty(self.N, dtype=dtype) for _ in range(self.nc)]
        u = np.empty((self.d, self.N), dtype=dtype) if want_u else None
        p = np.empty(self.N, dtype=dtype) if want_p else None
        ptrs = (C.c_void_p * self.nc)(*[r.ctypes.data for r in rho])
        self._check(self.L.lbm_get_macroscopic(self.h, ptrs, u.ctypes.data_as(C.c_void_p) if want_u else None,
                                               p.ctypes.data_as(C.c_void_p) if want_p else None, code, 0),
                    "lbm_get_macroscopic")
        return rho, u, p

    def get_macroscopic_device(self, want_u=True, want_p=True):
        """Device tensors in the compute dtype."""
        t = self.torch
        dt = self._ct_torch()
        rho = [t.empty(self.N, dtype=dt, device=self.device) for _ in range(self.nc)]
        u = t.empty((self.d, self.N), dtype=dt, device=self.device) if want_u else None
        p = t.empty(self.N, dtype=dt, device=self.device) if want_p else None
        ptrs = (C.c_void_p * self.nc)(*[r.data_ptr() for r in rho])
        self._check(self.L.lbm_get_macroscopic(self.h, ptrs, C.c_void_p(u.data_ptr()) if want_u else None,
                                               C.c_void_p(p.data_ptr()) if want_p else None,
                                               self.cfg.compute_dtype, 1), "lbm_get_macroscopic")
        return rho, u, p

    def get_populations(self, k: int = 0, dtype=np.float64) -> np.ndarray:
        code = DTYPES["f32"] if dtype == np.float32 else DTYPES["f64"]
        out = np.empty((self.q, self.N), dtype=dtype)
        self._check(self.L.lbm_get_populations(self.h, k, out.ctypes.data_as(C.c_void_p), code, 0), "lbm_get_populations")
        return out

    def get_populations_device(self, k: int = 0):
        out = self.torch.empty((self.q, self.N), dtype=self._ct_torch(), device=self.device)
        self._check(self.L.lbm_get_populations(self.h, k, C.c_void_p(out.data_ptr()), self.cfg.compute_dtype, 1),
                    "lbm_get_populations")
        return out

    def set_populations(self, k: int, f: np.ndarray):
        f = np.ascontiguousarray(f)
        assert f.shape == (self.q, self.N)
        self._check(self.L.lbm_set_populations(self.h, k, f.ctypes.data_as(C.c_void_p), _np_dtype_code(f), 0),
                    "lbm_set_populations")

    # ---- slab decomposition (include/lbm.h): packed halo layers as uint8 device tensors
    def halo_bytes(self, width: int) -> int:
        n = C.c_size_t(0)
        self._check(self.L.lbm_halo_bytes(self.h, int(width), C.byref(n)), "lbm_halo_bytes")
        return int(n.value)

    def export_halo(self, side: int, width: int, out=None):
        if out is None:
            out = self.torch.empty(self.halo_bytes(width), dtype=self.torch.uint8, device=self.device)
        assert out.is_cuda and out.is_contiguous() and out.numel() >= self.halo_bytes(width)
        self._check(self.L.lbm_export_halo(self.h, int(side), int(width), C.c_void_p(out.data_ptr())), "lbm_export_halo")
        return out

    def import_halo(self, side: int, width: int, buf):
        assert buf.is_cuda and buf.is_contiguous() and buf.numel() >= self.halo_bytes(width)
        self._check(self.L.lbm_import_halo(self.h, int(side), int(width), C.c_void_p(buf.data_ptr())), "lbm_import_halo")

    def get_link_flags(self) -> np.ndarray:
        out = np.empty(self.N, dtype=np.uint32)
        self._check(self.L.lbm_get_link_flags(self.h, out.ctypes.data_as(C.c_void_p), 0), "lbm_get_link_flags")
        return out

    def get_boundary_solids(self) -> np.ndarray:
        m = self.L.lbm_get_boundary_solids(self.h, None, 0)
        if m < 0:
            self._check(int(m), "lbm_get_boundary_solids")
        out = np.empty(m, dtype=np.int64)
        if m:
            self.L.lbm_get_boundary_solids(self.h, out.ctypes.data_as(C.c_void_p), m)
        return out

    def get_psi(self, k: int = 0, dtype=np.float64) -> np.ndarray:
        code = DTYPES["f32"] if dtype == np.float32 else DTYPES["f64"]
        out = np.empty(self.N, dtype=dtype)
        self._check(self.L.lbm_get_psi(self.h, k, out.ctypes.data_as(C.c_void_p), code, 0), "lbm_get_psi")
        return out

    def render_isosurface(self, iso: float, axis: int = 2, k: int = 0, dtype=np.float64):
        """(shade, depth) images [n_v, n_u] of the iso-surface rho^k = iso seen along +axis (include/lbm.h)."""
        code = DTYPES["f32"] if dtype == np.float32 else DTYPES["f64"]
        dims = [self.cfg.nx, self.cfg.ny, self.cfg.nz]
        nu, nv = [dims[a] for a in range(3) if a != axis][:2]    # a bad axis is the library's to reject
        shade = np.empty((nv, nu), dtype=dtype)
        depth = np.empty((nv, nu), dtype=dtype)
        self._check(self.L.lbm_render_isosurface(self.h, k, float(iso), int(axis), shade.ctypes.data_as(C.c_void_p),
                                                 depth.ctypes.data_as(C.c_void_p), code, 0), "lbm_render_isosurface")
        return shade, depth

    def set_profiling(self, enable: bool):
        self._check(self.L.lbm_set_profiling(self.h, 1 if enable else 0), "lbm_set_profiling")

    def get_kernel_times(self):
        """{kernel name: (total ms, launches)} since the last call (measurement only)."""
        ms = (C.c_double * len(KERNEL_IDS))()
        cnt = (C.c_int64 * len(KERNEL_IDS))()
        self._check(self.L.lbm_get_kernel_times(self.h, ms, cnt), "lbm_get_kernel_times")
        return {name: (ms[i], int(cnt[i])) for name, i in KERNEL_IDS.items()}

    @property
    def hot_path(self) -> str:
        """What the most recent step() launched: 'two_pass', 'one_pass_ws', 'one_pass_eq', 'two_pass_compact',
        'two_pass_persistent' or 'one_pass_tile'."""
        return {0: "none", 1: "two_pass", 3: "one_pass_ws", 4: "two_pass_compact", 5: "one_pass_eq",
                6: "two_pass_persistent", 7: "one_pass_tile"}[int(self.L.lbm_hot_path(self.h))]

    @property
    def steps_done(self) -> int:
        return int(self.L.lbm_steps_done(self.h))

    @property
    def kernel_launches(self) -> int:
        return int(self.L.lbm_kernel_launches(self.h))


def step_noalloc(wl: dict, f_in, f_out, stream=None) -> None:
    """lbm_step_noalloc (include/lbm.h): one time step f_in -> f_out on caller-held device tensors [nc][q][N] of the
    compute dtype (the arrays get_populations_device returns), with no handle, no workspace and no allocation: psi lives
    in a static device array inside the library (noalloc_max_scratch_bytes()).  Calls that overlap on the GPU race on it."""
    import torch
    L = load_library()
    cfg = make_config(wl)
    want = torch.float32 if wl.get("compute_dtype", "f64") == "f32" else torch.float64
    n = cfg.n_components * (9 if cfg.lattice == 0 else 19) * cfg.nx * cfg.ny * cfg.nz
    for t in (f_in, f_out):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == want and t.numel() == n):
            raise LBMError("step_noalloc: f_in / f_out must be contiguous CUDA tensors [nc][q][N] of the compute dtype")
    s = stream if stream is not None else torch.cuda.current_stream(f_in.device)
    with torch.cuda.device(f_in.device):
        rc = L.lbm_step_noalloc(C.byref(cfg), C.c_void_p(f_in.data_ptr()), C.c_void_p(f_out.data_ptr()), C.c_void_p(s.cuda_stream))
    if rc != LBM_OK:
        raise LBMError(f"lbm_step_noalloc failed: {STATUS.get(rc, rc)}: {L.lbm_noalloc_last_error().decode()}")


def noalloc_max_scratch_bytes() -> int:
    return int(load_library().lbm_noalloc_max_scratch_bytes())


def get_lattice(name: str):
    L = load_library()
    q = C.c_int(0)
    e = np.zeros((19, 3), dtype=np.int32)
    w = np.zeros(19, dtype=np.float64)
    opp = np.zeros(19, dtype=np.int32)
    rc = L.lbm_get_lattice(LATTICES[name], C.byref(q), e.ctypes.data_as(C.c_void_p), w.ctypes.data_as(C.c_void_p),
                           opp.ctypes.data_as(C.c_void_p))
    if rc != LBM_OK:
        raise LBMError("lbm_get_lattice failed")
    return e[: q.value].copy(), w[: q.value].copy(), opp[: q.value].copy()
