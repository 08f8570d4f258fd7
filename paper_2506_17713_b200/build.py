"""Build the CUDA C-ABI library in-tree: paper_2506_17713_b200/liblbm_b200.so (sm_100a).

nvcc cross-compiles without a GPU.  One object per translation unit, compiled in parallel.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
OBJ = HERE / "build"
LIB = HERE / "liblbm_b200.so"
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "--expt-relaxed-constexpr",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]
if os.environ.get("LBM_EXTRA_NVCC_FLAGS"):   # development switches, e.g. -DLBM_WS_TIMING
    FLAGS += os.environ["LBM_EXTRA_NVCC_FLAGS"].split()
if os.environ.get("LBM_FUSED_TUNING"):   # also build the K2F tile-shape experiments (lbm_launch.cuh)
    FLAGS.append("-DLBM_FUSED_TUNING")


def _newest_header() -> float:
    hs = list(CSRC.glob("*.cuh")) + list(CSRC.glob("*.h")) + [HERE.parent / "include" / "lbm.h"]
    return max(h.stat().st_mtime for h in hs)


def build(force: bool = False, verbose: bool = False, ptxas_v: bool = False) -> Path:
    OBJ.mkdir(exist_ok=True)
    # a change of compiler flags (development switches) rebuilds everything
    stamp = OBJ / "flags.txt"
    if not stamp.exists() or stamp.read_text() != " ".join(FLAGS):
        force = True
        stamp.write_text(" ".join(FLAGS))
    srcs = sorted(CSRC.glob("*.cu"))
    hdr = _newest_header()
    jobs = []
    for s in srcs:
        o = OBJ / (s.stem + ".o")
        if force or not o.exists() or o.stat().st_mtime < max(s.stat().st_mtime, hdr):
            jobs.append((s, o))

    def compile_one(job):
        s, o = job
        cmd = [NVCC, *FLAGS, "-c", str(s), "-o", str(o)]
        if ptxas_v:
            cmd += ["-Xptxas", "-v"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        return s, r

    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
            for s, r in ex.map(compile_one, jobs):
                if verbose or ptxas_v or r.returncode != 0:
                    sys.stderr.write(f"--- {s.name}\n{r.stdout}{r.stderr}\n")
                if r.returncode != 0:
                    raise RuntimeError(f"nvcc failed on {s.name}")
    objs = [str(OBJ / (s.stem + ".o")) for s in srcs]
    if jobs or not LIB.exists():
        cmd = [NVCC, "-shared", "-o", str(LIB), *objs, "-gencode", "arch=compute_100a,code=sm_100a", "-lcudart"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("link failed")
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose="-v" in sys.argv, ptxas_v="--ptxas" in sys.argv)
    print(LIB)
