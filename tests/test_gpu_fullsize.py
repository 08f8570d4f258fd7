"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default path, default dtypes).
The oracle cannot hold 512^3, so sampled cells are checked one by one: after K steps the populations of a cell depend
only on the initial state within a few cells per step, so the oracle runs K steps on a small periodic box cut out
around the sample (wrap-around extraction) and its centre cell is compared with the GPU's.  Plus properties that hold
at any size: total mass and, on the periodic domain, total momentum."""
import numpy as np
import pytest

from conftest import make_oracle
from paper_2506_17713_b200 import workloads as W
from test_gpu_parity import TOL32, make_gpu, with_dtype

pytestmark = pytest.mark.gpu

K = 3            # steps
R = 3 * K + 3    # half-width of the oracle's box: pull 1 + psi stencil 1 + virtual density 1 per step, and a margin


def cut(field, dims, centre, r):
    """(2r+1)^3 box around centre from a flat [N] field (x fastest), periodic wrap"""
    nx, ny, nz = dims
    f = np.asarray(field).reshape(nz, ny, nx)
    ix = [np.arange(c - r, c + r + 1) % n for c, n in zip(centre, (nx, ny, nz))]
    return f[np.ix_(ix[2], ix[1], ix[0])].reshape(-1)


def oracle_centre(wl, inp, dims, centre):
    m = 2 * R + 1
    sub = dict(wl, nx=m, ny=m, nz=m, periodic=(True, True, True))
    sub.pop("face_bc", None)
    sub.pop("path", None)
    sinp = dict(rho=[cut(r, dims, centre, R) for r in inp["rho"]], u=None,
                mask=None if inp.get("mask") is None else cut(inp["mask"], dims, centre, R))
    o = make_oracle(sub, sinp)
    o.step(K)
    c = R + m * (R + m * R)
    return [o.get_populations(k)[:, c] for k in range(wl["n_components"])]


def test_config5_512_sampled_cells_and_conservation():
    import torch
    n = 512
    wl, inp = W.config5(n, "f32")
    g = make_gpu(wl, inp)
    rho0 = torch.as_tensor(inp["rho"][0]).double().sum().item()
    g.step(K)
    torch.cuda.synchronize()
    assert g.hot_path == "one_pass_ws"
    f = g.get_populations_device(0)                                  # [19, N] on the device
    # properties: mass (exact up to fp32 rounding of 19 x 134 M values) and momentum (the Shan-Chen force sums to zero)
    mass = f.double().sum().item()
    assert abs(mass - rho0) <= 1e-6 * rho0
    from paper_2506_17713_b200 import binding
    e, w, opp = binding.get_lattice("D3Q19")
    mom = (torch.as_tensor(e, dtype=torch.float64, device=f.device).T @ f.double().sum(dim=1))
    assert mom.abs().max().item() <= 1e-6 * rho0
    # samples: interface cells (largest density jumps along x), tile seams of the one-pass kernel (x = 127|128, rows of 8,
    # the 128-plane chunks), the domain corners
    rho = np.asarray(inp["rho"][0]).reshape(n, n, n)
    jump = np.abs(np.diff(rho[::37, ::41, :], axis=2))
    zz, yy, xx = np.unravel_index(np.argsort(jump, axis=None)[-6:], jump.shape)
    samples = [(int(x), int(y) * 41, int(z) * 37) for x, y, z in zip(xx, yy, zz)]
    samples += [(0, 0, 0), (n - 1, n - 1, n - 1), (127, 7, 127), (128, 8, 128), (255, 511, 0), (384, 263, 383)]
    worst = 0.0
    for c in samples:
        fo = oracle_centre(with_dtype(wl, "f64"), inp, (n, n, n), c)[0]
        idx = c[0] + n * (c[1] + n * c[2])
        fg = f[:, idx].double().cpu().numpy()
        worst = max(worst, np.abs(fg - fo).max() / np.abs(fo).max())
    assert worst <= TOL32, worst


def test_config4_400_sampled_cells_compact_layout():
    import torch
    n = 400
    wl, inp = W.config4(n, store_dtype="f32")
    g = make_gpu(wl, inp)
    g.step(K)
    torch.cuda.synchronize()
    assert g.hot_path == "two_pass_compact"
    f = [g.get_populations_device(k) for k in range(2)]
    mask = np.asarray(inp["mask"]).reshape(n, n, n)
    # fluid cells next to solid cells (bounce-back links, virtual density), away from the inlet / outlet faces
    rng = np.random.default_rng(4)
    samples = []
    while len(samples) < 10:
        x, y, z = (int(v) for v in rng.integers(0, n, 3))
        if not (R + 1 <= x < n - R - 1) or mask[z, y, x]:
            continue
        if mask[z, y, x - 1] or mask[z, y, x + 1] or mask[z, (y + 1) % n, x] or mask[(z + 1) % n, y, x] or len(samples) >= 8:
            samples.append((x, y, z))
    worst = 0.0
    for c in samples:
        fo = oracle_centre(with_dtype(wl, "f64"), inp, (n, n, n), c)
        idx = c[0] + n * (c[1] + n * c[2])
        for k in range(2):
            fg = f[k][:, idx].double().cpu().numpy()
            worst = max(worst, np.abs(fg - fo[k]).max() / np.abs(fo[k]).max())
    assert worst <= TOL32, worst
    # the interior samples above never see the faces; the dense export of the whole state must still be finite
    assert all(bool(torch.isfinite(t).all()) for t in f)


@pytest.mark.parametrize("name", ["C3-256", "P4-416"])
def test_other_periodic_configs_at_full_size(name):
    """config 3 (MRT, Peng-Robinson) and the paper's own 416^3 case in the one-pass kernel, sampled like config 5"""
    import torch
    wl, inp = W.config3(256, "f32") if name == "C3-256" else W.paper_benchmark(416, "f32")
    n = wl["nx"]
    g = make_gpu(wl, inp)
    rho0 = torch.as_tensor(inp["rho"][0]).double().sum().item()
    g.step(K)
    torch.cuda.synchronize()
    assert g.hot_path == "one_pass_ws"
    f = g.get_populations_device(0)
    assert abs(f.double().sum().item() - rho0) <= 1e-6 * rho0
    rng = np.random.default_rng(11)
    samples = [(0, 0, 0), (n - 1, n - 1, n - 1), (127, 7, 127), (128, 8, 128), (n - 1, 0, n // 2)]
    samples += [tuple(int(v) for v in rng.integers(0, n, 3)) for _ in range(5)]
    if name == "P4-416":
        samples += [(n // 2 + 30, n // 2, n // 2), (n // 2, n // 2 - 30, n // 2), (n // 2 + 21, n // 2 + 21, n // 2)]   # droplet surface
    worst = 0.0
    for c in samples:
        fo = oracle_centre(with_dtype(wl, "f64"), inp, (n, n, n), c)[0]
        fg = f[:, c[0] + n * (c[1] + n * c[2])].double().cpu().numpy()
        worst = max(worst, np.abs(fg - fo).max() / np.abs(fo).max())
    assert worst <= TOL32, worst
