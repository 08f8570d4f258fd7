"""lbm_step_noalloc (include/lbm.h): the time step for callers that cannot allocate -- no handle, no workspace, psi in a
static device array inside the library.  Checked against the resident path (lbm_create + lbm_step) on the same populations,
two calls in a row (the second call finds the first call's psi in the scratch array, and a larger domain's before that),
within the tolerances of test_gpu_parity.py.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_2506_17713_b200 import workloads as W
from test_gpu_parity import TOL32, TOL64, make_gpu, small_inputs

pytestmark = pytest.mark.gpu


def _cases():
    c1, i1 = W.config1(64, "f64")                                   # D2Q9, one component, CS EOS, BGK, fp64
    c3, _ = W.config3(24, "f32")                                    # D3Q19, Peng-Robinson, MRT, fp32
    c2, _ = W.config2(96, 64, "f32")                                # D2Q9, two components (no plates here: fully periodic)
    c5, _ = W.config5(16, "f64")
    c5.update(nx=40, ny=12, nz=9, forcing="SHIFT", tau=[0.8], body_accel=(1e-5, 0.0, -2e-5))   # BGK tau != 1, shift forcing, body force
    return [("C1-64-f64", c1, dict(rho=i1["rho"], u=None, mask=None)),
            ("C3-24-f32-mrt", c3, small_inputs(c3, 3, 0.05, 0.3)),
            ("C2-96x64-f32-2comp", c2, small_inputs(c2, 4, 0.1, 0.9)),
            ("C5-40x12x9-f64-shift", c5, small_inputs(c5, 5, 0.05, 0.3))]


def _compare(a, b, wl):
    a, b = a.cpu().numpy().astype(np.float64), b.cpu().numpy().astype(np.float64)
    assert np.isfinite(b).all()
    if wl["compute_dtype"] == "f64":
        assert np.abs(a - b).max() <= TOL64, np.abs(a - b).max()
    else:
        assert np.abs(a - b).max() <= TOL32 * np.abs(a).max(), (np.abs(a - b).max(), np.abs(a).max())


def test_step_noalloc_matches_the_resident_path_two_calls_in_a_row():
    import torch
    from paper_2506_17713_b200 import binding
    assert binding.noalloc_max_scratch_bytes() == 2 << 20
    # a call on the largest case first, so that every later call finds foreign psi values in the scratch array
    for name, wl, inp in sorted(_cases(), key=lambda c: -c[1]["nx"] * c[1]["ny"] * c[1]["nz"] * c[1]["n_components"]):
        g = make_gpu(dict(wl, path="two_pass"), inp)
        nc = wl["n_components"]
        pops = lambda: torch.stack([g.get_populations_device(k) for k in range(nc)]).contiguous()
        f0 = pops()
        g.step(1)
        f1 = pops()
        g.step(1)
        f2 = pops()
        h1, h2 = torch.empty_like(f0), torch.empty_like(f0)
        binding.step_noalloc(wl, f0, h2)          # (the first call of a kernel may load its code: not counted below)
        torch.cuda.synchronize()
        free = torch.cuda.mem_get_info()[0]
        binding.step_noalloc(wl, f0, h1)          # two calls in a row on the same stream: ordered, no race on the scratch
        binding.step_noalloc(wl, h1, h2)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free          # nothing was allocated on the device
        _compare(f1, h1, wl)
        _compare(f2, h2, wl)
        # mass of every component is conserved by the step (periodic, no solids): an independent sanity check
        q = f0.shape[1]
        for k in range(nc):
            m0, m2 = f0[k].double().sum().item(), h2[k].double().sum().item()
            assert abs(m2 - m0) <= (1e-12 if wl["compute_dtype"] == "f64" else 2e-6) * abs(m0) * q


def test_step_noalloc_refuses_what_it_cannot_hold_or_does_not_build():
    import torch
    from paper_2506_17713_b200 import binding
    big, _ = W.config5(96, "f32")                                   # 96^3 * 4 B = 3.4 MiB of psi > 2 MiB
    cfg = binding.make_config(big)
    import ctypes as C
    L = binding.load_library()
    rc = L.lbm_step_noalloc(C.byref(cfg), C.c_void_p(256), C.c_void_p(512), None)   # pointers never touched: the size check comes first
    assert rc == -3 and b"static scratch array holds 2097152" in L.lbm_noalloc_last_error()
    ok, inp = W.config1(32, "f64")
    g = make_gpu(ok, dict(rho=inp["rho"], u=None, mask=None))
    f0 = g.get_populations_device(0).unsqueeze(0).contiguous()
    with pytest.raises(binding.LBMError, match="distinct"):
        binding.step_noalloc(ok, f0, f0)                            # in place: the push would race with the reads
    with pytest.raises(binding.LBMError, match="periodic"):
        binding.step_noalloc(dict(ok, periodic=(True, False, True)), f0, torch.empty_like(f0))
    out = torch.empty_like(f0)
    binding.step_noalloc(ok, f0, out)                               # and still works after the refusals
    g.step(1)
    torch.cuda.synchronize()
    _compare(g.get_populations_device(0).unsqueeze(0), out, ok)
