"""CPU-side checks of the C-ABI boundary: the library builds for sm_100a, loads, exports every
symbol include/lbm.h declares, and its host-only entry points behave.  No kernel is launched."""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    from paper_2506_17713_b200 import build as b
    b.build()
    from paper_2506_17713_b200 import binding
    return binding


def _declared_symbols():
    text = (ROOT / "include" / "lbm.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lbm_[a-z_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    L = lib.load_library()
    names = _declared_symbols()
    assert {"lbm_create", "lbm_set_solid_mask", "lbm_init_fields", "lbm_step", "lbm_get_macroscopic",
            "lbm_workspace_bytes", "lbm_set_face_bc", "lbm_get_populations", "lbm_get_link_flags",
            "lbm_destroy"} <= set(names)
    for n in names:
        assert hasattr(L, n), n
    assert set(names) == set(lib._SIGNATURES)  # the binding mirrors the header one to one


def test_config_struct_layout(lib):
    assert lib.load_library().lbm_config_bytes() == C.sizeof(lib.lbm_config_t)


def test_lattice_tables_match_oracle(lib):
    """Direction order is part of the ABI; the CUDA path's own tables must agree with the oracle's."""
    from oracle import lbm_oracle as o
    for name in ("D2Q9", "D3Q19"):
        e, w, opp = lib.get_lattice(name)
        eo, wo, oppo = o.lattice(name)
        assert np.array_equal(e, eo)
        assert np.allclose(w, wo, rtol=0, atol=1e-16)
        assert np.array_equal(opp, oppo)


def test_workspace_bytes_and_invalid_configs(lib):
    from paper_2506_17713_b200 import workloads as W
    L = lib.load_library()
    wl, _ = W.config5(64)
    cfg = lib.make_config(wl)
    nbytes = L.lbm_workspace_bytes(C.byref(cfg))
    N = 64 ** 3
    assert nbytes >= 2 * 19 * N * 4 + 2 * N * 4
    assert nbytes < 8 * 19 * N * 4
    bad = lib.make_config(wl)
    bad.nx = 0
    assert L.lbm_workspace_bytes(C.byref(bad)) == 0
    bad = lib.make_config(wl)
    bad.G[0][0] = 1.0       # EOS psi needs g_kk < 0 (reading R4)
    assert L.lbm_workspace_bytes(C.byref(bad)) == 0
    bad = lib.make_config(wl)
    bad.compute_dtype, bad.store_dtype = lib.DTYPES["f64"], lib.DTYPES["f16"]
    assert L.lbm_workspace_bytes(C.byref(bad)) == 0
    # create without a workspace is refused before anything touches a device
    h = C.c_void_p()
    assert L.lbm_create(C.byref(cfg), None, 0, None, C.byref(h)) == -3   # LBM_E_NOMEM
    assert not h.value
    assert L.lbm_version().startswith(b"paper_2506_17713_b200")


def test_no_cpu_fallback(lib):
    """Without a CUDA device the product path refuses to run (it never routes through the oracle)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2506_17713_b200 import workloads as W
    wl, _ = W.config1(16)
    with pytest.raises(lib.LBMError):
        lib.LBM(wl)
    src = (ROOT / "paper_2506_17713_b200" / "binding.py").read_text()
    assert "oracle" not in src.replace("(it never routes through the oracle)", "")
