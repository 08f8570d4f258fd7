#!/usr/bin/env python
"""bench.py -- MLUPS of the Shan-Chen LBM hot path on B200 (metric of BASELINE.json).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5-512] [--impl ours|reference]

A "step" is ONE lattice time step = one pass of the whole hot path (S1..S7 of DESIGN.md: moments, psi,
virtual density, force, collide, stream + boundaries) over the whole synthetic domain.  MLUPS follows the
paper's Eq. 24: n_components * nx*ny*nz * steps / (t * 1e6).

What is printed (ONE JSON line on rank 0):
  value      whole-job MLUPS with the populations already resident in HBM (CUDA events on the launch stream,
             barrier + synchronize on both sides, max over ranks)
  e2e        the same metric through the C-ABI with HOST buffers: lbm_init_fields(pinned host rho) ->
             lbm_step(K) -> lbm_get_macroscopic(pinned host rho); both copies inside the timed region
  roofline   dominant kernel: algorithmic bytes per launch / its average launch time, measured live with
             CUDA event pairs recorded by the library on its own stream (lbm_set_profiling), against
             MEASURED_PEAKS.json's hbm_gbs
  cpu_baseline  the oracle (oracle/, as it stands) timed on this box's host cores on a bounded sample
  configs    (--all-configs, default on at N=1) MLUPS of the other BASELINE.json configs, short runs

--impl reference times the oracle alone (there is no reference implementation of the paper to install;
the oracle is the reference arm for this tier).  N > 1: the path is built for one GPU (north_star), so
--gpus N runs N independent replicas, one per rank ("replicas only").
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

from paper_2506_17713_b200 import workloads as W  # noqa: E402  (seeded inputs only: no arithmetic of the method)

DT_BYTES = {"f16": 2, "f32": 4, "f64": 8}


# --------------------------------------------------------------------------- workloads
def make_workload(name: str):
    """name = C<config>-<size>[-<variant>] ; returns (workload dict, inputs)."""
    parts = name.split("-")
    cfg, size = parts[0].upper(), int(parts[1]) if len(parts) > 1 else None
    var = parts[2] if len(parts) > 2 else None
    if cfg == "C1":
        return W.config1(size or 64, var or "f64")
    if cfg == "C2":
        n = size or 512
        return W.config2(n, n // 2, var or "f32")
    if cfg == "C3":
        return W.config3(size or 256, var or "f32")
    if cfg == "C4":
        return W.config4(size or 400, store_dtype=var or "f16")
    if cfg == "C5":
        return W.config5(size or 512, var or "f32")
    if cfg == "P4":
        return W.paper_benchmark(size or 416, var or "f32")
    raise SystemExit(f"unknown workload {name}")


def algorithmic_bytes(wl, kernel: str, path: str = "") -> float:
    """Algorithmic bytes per component-cell update of one kernel (
    SURVEY.md 8(d)): q populations of s store bytes, scalars of c compute bytes.  On the fluid-compact path
    (path = "two_pass_compact") K2 also reads its neighbour table (4 (q-1) bytes per fluid cell) and K1 writes rho."""
    q = 9 if wl["lattice"] == "D2Q9" else 19
    s = DT_BYTES[wl["store_dtype"]]
    c = DT_BYTES[wl["compute_dtype"]]
    nc = wl["n_components"]
    compact = path == "two_pass_compact"
    if kernel == "moments":   # K1: read q*s, write psi (+ rho for K1b)
        return q * s + c + (c if compact else 0)
    if kernel == "virtual":   # K1b: per boundary solid, not per cell: counted in path_bytes only
        return 0.0
    if kernel == "step":      # K2: read q*s + psi + mask bits (or the table), write q*s
        return 2 * q * s + c + (4.0 * (q - 1) / nc if compact else 0.25 / nc)
    if kernel == "fused":     # K2F: read q*s, write q*s (+ mask bits)
        return 2 * q * s + 0.125 / nc
    if kernel == "persistent":  # small domains: all steps of a call in one launch; per step the bytes of the path it runs
        return 2 * q * s + 0.25 / nc if path == "one_pass_tile" else 3 * q * s + 2 * c + 0.25 / nc
    if kernel == "two_pass":  # B2 of SURVEY 8(d)
        return 3 * q * s + 2 * c + 0.25 / nc
    raise KeyError(kernel)


def path_bytes(wl, path: str) -> float:
    """Algorithmic bytes per component-cell update of the whole step ON THE PATH THAT RAN (lbm_hot_path): B1 for the
    one-pass kernels, B2 for the two-pass path, B2 + rho + table for the fluid-compact path."""
    if path.startswith("one_pass"):
        return algorithmic_bytes(wl, "fused")
    return algorithmic_bytes(wl, "moments", path) + algorithmic_bytes(wl, "step", path)


# --------------------------------------------------------------------------- clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period=0.1):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.stop_flag = [], set(), threading.Event()
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            # CUDA_VISIBLE_DEVICES may remap; use the PCI bus id of the torch device
            import torch
            bus = torch.cuda.get_device_properties(index).pci_bus_id if hasattr(
                torch.cuda.get_device_properties(index), "pci_bus_id") else None
            self.h = None
            if bus is not None:
                for i in range(pynvml.nvmlDeviceGetCount()):
                    hh = pynvml.nvmlDeviceGetHandleByIndex(i)
                    if pynvml.nvmlDeviceGetPciInfo(hh).bus == bus:
                        self.h = hh
            if self.h is None:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self.stop_flag.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def result(self):
        self.stop_flag.set()
        if self.is_alive():
            self.join(timeout=2)
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# --------------------------------------------------------------------------- oracle timing (CPU)
def time_oracle(sample_name: str, steps: int, warmup: int, budget_s: float = 20.0, threads: int = 0):
    """Times the oracle as it stands (OpenMP over the outer loops; threads = 0: all host cores) on a bounded sample."""
    from oracle import lbm_oracle

    lbm_oracle.build()
    cores = lbm_oracle.set_threads(threads if threads > 0 else lbm_oracle.host_cores())
    wl, inp = make_workload(sample_name)
    o = lbm_oracle.Oracle(wl)
    if inp.get("mask") is not None:
        o.set_solid_mask(inp["mask"])
    o.init_fields(inp["rho"])
    t0 = time.perf_counter()
    o.step(max(1, warmup))
    per = (time.perf_counter() - t0) / max(1, warmup)
    if steps <= 0:
        steps = int(max(2, min(200, budget_s / max(per, 1e-6))))
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    cells = wl["nx"] * wl["ny"] * wl["nz"] * wl["n_components"]
    if wl["nx"] * wl["ny"] * wl["nz"] < 262144:
        cores = 1   # the oracle's loops go parallel from 262 144 cells up (oracle/lbm_oracle.cpp): one thread did the work
    return dict(value=cells * steps / dt / 1e6, unit="MLUPS", cores=cores, kind="oracle",
                sample=f"{sample_name}: {wl['lattice']} {wl['nx']}x{wl['ny']}x{wl['nz']} n_c={wl['n_components']} "
                       f"{wl['collision']} {wl['compute_dtype']}/{wl['store_dtype']}, {steps} steps after "
                       f"{max(1, warmup)} warm-up, OpenMP {cores} threads",
                steps=steps, ms_per_step=dt / steps * 1e3), wl


def cpu_sample_of(workload: str) -> str:
    """Bounded CPU sample of a workload: the same recipe at a size the oracle steps in ~0.1-1 s."""
    parts = workload.split("-")
    cfg = parts[0].upper()
    size = int(parts[1]) if len(parts) > 1 else None
    cap = {"C1": 64, "C2": 512, "C3": 96, "C4": 96, "C5": 128, "P4": 128}[cfg]
    n = min(size or cap, cap)
    return "-".join([cfg, str(n)] + parts[2:])


# --------------------------------------------------------------------------- GPU runs
def gpu_run(torch, workload: str, steps: int, warmup: int, dist, want_roofline=True, want_e2e=True, device=0):
    from paper_2506_17713_b200 import binding

    wl, inp = make_workload(workload)
    nc = wl["n_components"]
    N = wl["nx"] * wl["ny"] * wl["nz"]
    np_dt = np.float32 if wl["compute_dtype"] == "f32" else np.float64
    stream = torch.cuda.Stream(device=device)
    sim = binding.LBM(wl, device=f"cuda:{device}", stream=stream)
    if inp.get("mask") is not None:
        sim.set_solid_mask(inp["mask"])
    # pinned host inputs (used by the e2e leg) and the same arrays for the resident leg
    host_rho = [torch.from_numpy(np.ascontiguousarray(r, dtype=np_dt)).pin_memory() for r in inp["rho"]]
    host_out = [torch.empty(N, dtype=host_rho[0].dtype).pin_memory() for _ in range(nc)]
    sim.init_fields([h.numpy() for h in host_rho])

    def barrier():
        torch.cuda.synchronize(device)
        if dist is not None:
            dist.barrier()

    # ---- resident leg: K steps, device timing on the launch stream
    sim.step(warmup)
    barrier()
    l0 = sim.kernel_launches
    sampler = ClockSampler(device)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    sim.step(steps)
    e1.record(stream)
    barrier()
    clocks = sampler.result()
    ms = e0.elapsed_time(e1)
    launches = sim.kernel_launches - l0
    out = dict(wl=wl, N=N, ms=ms, launches=launches, clocks=clocks, path=sim.hot_path)

    # ---- per-kernel leg (roofline numerator): library-recorded event pairs on its own stream
    if want_roofline:
        sim.set_profiling(True)
        sim.get_kernel_times()
        sim.step(min(steps, 50))
        out["kernel_times"] = sim.get_kernel_times()
        sim.set_profiling(False)

    # ---- e2e leg: host rho -> K steps -> host rho, copies inside the timed region
    if want_e2e:
        ksteps = steps

        def job():
            sim.init_fields([h.numpy() for h in host_rho])
            sim.step(ksteps)
            ptrs = (binding.C.c_void_p * nc)(*[h.data_ptr() for h in host_out])
            sim._check(sim.L.lbm_get_macroscopic(sim.h, ptrs, None, None, binding.DTYPES[wl["compute_dtype"]], 0),
                       "lbm_get_macroscopic")

        job()  # warm-up job
        barrier()
        t0 = time.perf_counter()
        e0.record(stream)
        job()
        e1.record(stream)
        barrier()
        wall = (time.perf_counter() - t0) * 1e3
        out["e2e_ms"] = max(e0.elapsed_time(e1), wall)  # host-side staging syncs are part of the job
        out["e2e_steps"] = ksteps
        out["h2d"] = sum(h.numel() * h.element_size() for h in host_rho)
        out["d2h"] = sum(h.numel() * h.element_size() for h in host_out)
        out["mass_out"] = float(sum(h.double().sum().item() for h in host_out))
    sim.close()
    return out


def make_roofline(workload: str, r: dict, mlups: float, peak: float, peak_src: str):
    """The `roofline` object of one GPU run: the dominant kernel's algorithmic bytes per launch over its average launch
    time (library-recorded event pairs), against the measured copy bandwidth.  Bytes are those of the path that ran."""
    wl, N, kt, path = r["wl"], r["N"], r.get("kernel_times", {}), r.get("path", "")
    nc = wl["n_components"]
    kt = {k: v for k, v in kt.items() if v[1] > 0}
    if not kt:
        return None
    dom = max(kt, key=lambda k: kt[k][0])
    avg_ms = kt[dom][0] / kt[dom][1]
    ff = wl.get("fluid_fraction", 1.0)    # config 4: solid cells move no populations
    per_update = algorithmic_bytes(wl, dom, path)
    ach = per_update * nc * N * ff / (avg_ms * 1e-3) / 1e9
    tot = sum(v[0] for v in kt.values())
    out = {"bound": "hbm", "kernel": dom, "path": path, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
           "traffic": None, "peak_source": peak_src, "avg_launch_ms": avg_ms,
           "algorithmic_bytes_per_update": per_update,
           "units_per_launch": nc * N * ff,
           "kernel_share_of_step": kt[dom][0] / tot if tot > 0 else None,
           "kernels_ms_per_step": {k: v[0] / max(1, kt[dom][1]) for k, v in kt.items()},
           # whole step on the bytes of the path that ran, against the measured copy bandwidth
           "step_bytes_per_update": path_bytes(wl, path),
           "step_frac_of_measured": mlups * ff * path_bytes(wl, path) * 1e6 / (peak * 1e9),
           # north_star's contract number (SURVEY 8(d) "graded"): two-pass bytes B2 against the nominal 8 TB/s, whatever
           # path ran -- NOT an achieved bandwidth (the one-pass kernels move B1 < B2 bytes)
           "north_star_frac_B2_of_8TBs": mlups * ff * algorithmic_bytes(wl, "two_pass") * 1e6 / 8e12}
    tf = ROOT / "profiles" / "traffic.json"   # per-launch DRAM bytes from the committed ncu --set full captures
    if tf.exists():
        try:
            out["traffic"] = json.loads(tf.read_text()).get(f"{workload}:{dom}")
        except Exception:
            pass
    return out


def l2_note(wl, nc, N) -> str:
    """Timing rule: inputs larger than L2, or say that the workload itself lives in L2."""
    gb = 2 * nc * (9 if wl["lattice"] == "D2Q9" else 19) * N * DT_BYTES[wl["store_dtype"]] / 1e9
    if gb > 0.5:
        return "populations (%.1f GB) larger than L2, no flush needed" % gb
    return ("populations (%.1f MB) smaller than L2: consecutive time steps of one domain, L2-resident by nature of the "
            "workload (the roofline fraction against HBM is context only; the step is latency-bound)" % (gb * 1e3))


def reduce_max(torch, dist, x: float) -> float:
    if dist is None:
        return x
    t = torch.tensor([x], dtype=torch.float64, device="cuda" if torch.cuda.is_available() else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C5-512", help="C<config>-<size>[-variant], e.g. C5-512, C3-256, C4-400-f16")
    ap.add_argument("--all-configs", dest="all_configs", action="store_true", default=None)
    ap.add_argument("--no-all-configs", dest="all_configs", action="store_false")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    # ------------------------------------------------------------------ reference arm = the oracle on host cores
    if args.impl == "reference":
        if rank != 0:
            return 0
        sample = cpu_sample_of(args.workload)
        res, wl = time_oracle(sample, args.steps if args.steps < 200 else 0, args.warmup)
        line = {
            "impl": "reference", "metric": "MLUPS", "value": res["value"], "unit": "MLUPS", "n_gpus": args.gpus,
            "steps": res["steps"], "warmup": args.warmup, "ms_per_step": res["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": wl["compute_dtype"], "data": "synthetic",
            "config": {"workload": args.workload, "sample": sample, "note": "oracle (plain C++ loops written from the "
                       "paper) on host cores; a bounded sample of the workload; not a GPU number"},
            "cpu_baseline": {k: res[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": res["value"], "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0,
        }
        print(json.dumps(line))
        return 0

    # ------------------------------------------------------------------ our arm
    import torch

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the LBM path has no CPU fallback")
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        torch.cuda.set_device(local_rank)
        dist_mod.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
        dist = dist_mod
    device = local_rank if world > 1 else 0
    torch.cuda.set_device(device)

    r = gpu_run(torch, args.workload, args.steps, args.warmup, dist, device=device)
    wl, N = r["wl"], r["N"]
    nc = wl["n_components"]
    ms = reduce_max(torch, dist, r["ms"])
    value = world * nc * N * args.steps / (ms * 1e-3) / 1e6
    e2e_ms = reduce_max(torch, dist, r["e2e_ms"])
    e2e_value = world * nc * N * r["e2e_steps"] / (e2e_ms * 1e-3) / 1e6

    peaks_file = ROOT / "MEASURED_PEAKS.json"
    if peaks_file.exists():
        peak, peak_src = float(json.loads(peaks_file.read_text())["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    else:
        peak, peak_src = 6650.0, "fallback 6.65 TB/s of B200_PROFILING.md (of fallback)"
    roofline = make_roofline(args.workload, r, value / world, peak, peak_src)

    line = {
        "metric": "MLUPS", "value": value, "unit": "MLUPS", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": wl["compute_dtype"], "data": "synthetic",
        "config": {"workload": args.workload, "lattice": wl["lattice"], "grid": [wl["nx"], wl["ny"], wl["nz"]],
                   "n_components": nc, "collision": wl["collision"], "forcing": wl["forcing"], "psi": wl["psi_kind"],
                   "compute_dtype": wl["compute_dtype"], "store_dtype": wl["store_dtype"],
                   "parallelism": "single GPU" if world == 1 else f"{world} independent replicas",
                   "l2": l2_note(wl, nc, N)},
        "clocks": r["clocks"],
        "e2e": {"value": e2e_value, "unit": "MLUPS", "h2d_bytes_per_step": r["h2d"] / r["e2e_steps"],
                "d2h_bytes_per_step": r["d2h"] / r["e2e_steps"], "steps_per_call": r["e2e_steps"],
                "h2d_bytes_per_call": r["h2d"], "d2h_bytes_per_call": r["d2h"],
                "what": "lbm_init_fields(pinned host rho) + lbm_step(K) + lbm_get_macroscopic(pinned host rho), one call each"},
        "gpu_launches": r["launches"],
        "hot_path": r["path"],
        "roofline": roofline,
    }

    if rank == 0 and world == 1:
        def cpu_pair(workload, budget):
            """The oracle on this box's host cores, single-threaded and with OpenMP on all cores, on the
            bounded CPU sample of the workload."""
            sample = cpu_sample_of(workload)
            one, _ = time_oracle(sample, 0, 1, budget_s=budget, threads=1)
            allc, _ = time_oracle(sample, 0, 1, budget_s=budget, threads=0)
            return one, allc

        if not args.no_cpu_baseline:
            print("[bench] cpu baseline ...", file=sys.stderr, flush=True)
            one, allc = cpu_pair(args.workload, 8.0)
            line["cpu_baseline"] = {k: allc[k] for k in ("value", "unit", "cores", "kind", "sample")}
            line["cpu_baseline"]["single_thread"] = {"value": one["value"], "unit": "MLUPS", "cores": 1}
        if args.all_configs is None or args.all_configs:
            others = {}
            for name, k in (("C1-64", 2000), ("C2-512", 2000), ("C3-256", 100), ("C4-400-f16", 50), ("C4-400-f32", 50),
                            ("C5-128", 500), ("C5-256", 200), ("C5-384", 100), ("C5-256-f64", 100),
                            ("P4-416", 100)):   # the paper's own benchmark case, SURVEY 8(f) rank 4
                try:
                    print(f"[bench] {name} ...", file=sys.stderr, flush=True)
                    rr = gpu_run(torch, name, k, 10, None, want_roofline=True, want_e2e=False)
                    w2 = rr["wl"]
                    mlups = w2["n_components"] * rr["N"] * k / (rr["ms"] * 1e-3) / 1e6
                    ent = {"MLUPS": mlups, "ms_per_step": rr["ms"] / k, "path": rr["path"],
                           "roofline": make_roofline(name, rr, mlups, peak, peak_src)}
                    if "fluid_fraction" in w2:   # config 4: graded on fluid-cell updates
                        ent["porosity"] = w2["porosity"]
                        ent["fluid_fraction"] = w2["fluid_fraction"]
                        ent["fluid_MLUPS"] = mlups * w2["fluid_fraction"]
                    if not args.no_cpu_baseline and name in ("C1-64", "C2-512", "C3-256", "C4-400-f32", "P4-416"):
                        one, allc = cpu_pair(name, 2.5)
                        ent["cpu_baseline"] = {"sample": allc["sample"], "openmp": {"value": allc["value"], "cores": allc["cores"]},
                                               "single_thread": {"value": one["value"], "cores": 1}, "unit": "MLUPS", "kind": "oracle"}
                    others[name] = ent
                except Exception as ex:  # a config that does not fit / fails must not hide the headline
                    others[name] = {"error": repr(ex)[:200]}
            line["configs"] = others
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
