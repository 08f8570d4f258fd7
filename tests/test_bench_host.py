"""Host-side logic of bench.py (no GPU): roofline byte counts, workload naming, the reference arm's JSON contract and
the max-over-ranks reduction of the N > 1 path (world_size 2 over gloo; the path itself is "replicas only")."""
import json
import os
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))
import bench  # noqa: E402


def test_algorithmic_bytes_match_design_table():
    wl = dict(lattice="D3Q19", store_dtype="f32", compute_dtype="f32", n_components=1)
    assert bench.algorithmic_bytes(wl, "moments") == 80
    assert bench.algorithmic_bytes(wl, "step") == 156.25
    assert bench.algorithmic_bytes(wl, "two_pass") == 3 * 76 + 2 * 4 + 0.25    # B2 = 3 q s + 2 c + 0.25 / n_c
    assert bench.algorithmic_bytes(wl, "fused") == 152.125
    wl16 = dict(lattice="D3Q19", store_dtype="f16", compute_dtype="f32", n_components=2)
    assert bench.algorithmic_bytes(wl16, "two_pass") == 3 * 19 * 2 + 8 + 0.125
    wl2d = dict(lattice="D2Q9", store_dtype="f64", compute_dtype="f64", n_components=1)
    assert bench.algorithmic_bytes(wl2d, "two_pass") == 3 * 72 + 2 * 8 + 0.25


def test_workload_names_and_cpu_samples():
    wl, inp = bench.make_workload("C1-64")
    assert (wl["lattice"], wl["nx"], wl["ny"], wl["compute_dtype"]) == ("D2Q9", 64, 64, "f64")
    assert len(inp["rho"]) == 1 and inp["rho"][0].size == 64 * 64
    wl, _ = bench.make_workload("C5-32-f64")
    assert (wl["nx"], wl["compute_dtype"]) == (32, "f64")
    assert bench.cpu_sample_of("C5-512") == "C5-128"
    assert bench.cpu_sample_of("C4-400-f16") == "C4-96-f16"
    assert bench.cpu_sample_of("C1-64") == "C1-64"


def _run_reference(rank, world):
    env = dict(os.environ, RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), OMP_NUM_THREADS="2")
    return subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", str(world), "--workload", "C1-64",
                           "--steps", "3", "--warmup", "3"], capture_output=True, text=True, env=env, timeout=300)


def test_reference_arm_contract_rank0_prints_other_ranks_exit():
    r0 = _run_reference(0, 2)
    assert r0.returncode == 0, r0.stderr
    line = json.loads([l for l in r0.stdout.splitlines() if l.startswith("{")][-1])
    assert line["impl"] == "reference" and line["metric"] == "MLUPS" and line["unit"] == "MLUPS"
    assert line["value"] > 0 and line["higher_is_better"] is True and line["n_gpus"] == 2
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == {"value": line["value"], "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    r1 = _run_reference(1, 2)
    assert r1.returncode == 0 and r1.stdout.strip() == ""


def _gloo_worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.reduce_max(torch, dist, 1.5 + rank)      # every rank must see the slowest rank's time
    dist.barrier()
    out.put((rank, ms))
    dist.destroy_process_group()


def test_max_over_ranks_world_size_2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got == {0: 2.5, 1: 2.5}
