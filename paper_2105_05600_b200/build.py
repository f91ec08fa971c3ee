"""In-tree build of the C-ABI CUDA library (sm_100a only).  `python -m paper_2105_05600_b200.build`."""
from __future__ import annotations

import os
import shutil
import subprocess
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "librosefusion_b200.so"
SOURCES = ["rf_volume.cu", "rf_integrate.cu", "rf_atlas.cu", "rf_fitness.cu", "rf_track.cu", "rf_raycast.cu", "rf_surface.cu", "rf_gn.cu", "rf_baselines.cu", "rf_microbench.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: cannot build librosefusion_b200.so")


def stale() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    deps = [CSRC / s for s in SOURCES] + [CSRC / "rf_common.cuh", PKG.parent / "include" / "rosefusion_b200.h"]
    return any(d.stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not stale():
        return LIB
    tmp = LIB.with_suffix(f".{os.getpid()}.tmp")
    # RF_NVCC_EXTRA: extra nvcc flags for debug / tuning builds, e.g. "-DRF_CHECK_INSIDE" (k_update verifies k_cull's claims per voxel)
    extra = os.environ.get("RF_NVCC_EXTRA", "").split()
    cmd = [_nvcc(), *NVCC_FLAGS, *extra, "-o", str(tmp), *[str(CSRC / s) for s in SOURCES]]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
