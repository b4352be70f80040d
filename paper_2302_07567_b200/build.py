"""Build libfmm_b200.so (the C-ABI library of include/fmm.h) in-tree with nvcc for sm_100a.

``python -m paper_2302_07567_b200.build`` or ``build_library()``.  nvcc cross-compiles without a GPU.
The objects go to ``csrc/build/`` (git-ignored); the library sits next to this file so that it travels
with the source tree.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
LIB = HERE / "libfmm_b200.so"
PROBE_LIB = HERE / "libfmm_probe.so"   # FP64 pipe micro-benchmarks for bench.py (measurement tooling, not the boundary)
SOURCES = ["fmm_api.cu", "sort.cu", "kernels_tree.cu", "kernels_kd.cu", "kernels_dtt.cu", "kernels_interp.cu", "kernels_pairs.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: libfmm_b200.so cannot be built")
    return exe


def _newest_dep() -> float:
    deps = list(CSRC.glob("*.cu")) + list(CSRC.glob("*.cuh")) + [HERE.parent / "include" / "fmm.h", Path(__file__)]
    return max(p.stat().st_mtime for p in deps)


def build_library(force: bool = False, verbose: bool = False) -> Path:
    if not force and LIB.exists() and LIB.stat().st_mtime >= _newest_dep():
        return LIB
    nvcc = _nvcc()
    objdir = CSRC / "build"
    objdir.mkdir(exist_ok=True)

    def compile_one(src: str):
        obj = objdir / (src[:-3] + ".o")
        cmd = [nvcc, *NVCC_FLAGS, "-c", str(CSRC / src), "-o", str(obj)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        (objdir / (src[:-3] + ".ptxas.log")).write_text(r.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{r.stderr}")
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
    cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", str(tmp), *map(str, objs)]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stderr}")
    os.replace(tmp, LIB)
    if verbose:
        print(f"built {LIB}")
    return LIB


def build_probe(force: bool = False) -> Path:
    """libfmm_probe.so from csrc/probe_fp64.cu (see the header comment of that file)."""
    src = CSRC / "probe_fp64.cu"
    if not force and PROBE_LIB.exists() and PROBE_LIB.stat().st_mtime >= src.stat().st_mtime:
        return PROBE_LIB
    tmp = PROBE_LIB.with_suffix(f".tmp{os.getpid()}.so")
    cmd = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
           "-shared", str(src), "-o", str(tmp)]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on probe_fp64.cu:\n{r.stderr}")
    os.replace(tmp, PROBE_LIB)
    return PROBE_LIB


if __name__ == "__main__":
    build_library(force="--force" in sys.argv, verbose=True)
    build_probe(force="--force" in sys.argv)
