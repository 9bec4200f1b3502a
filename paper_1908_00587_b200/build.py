"""Builds ``libnsc.so`` (the C-ABI library of include/nsc.h) in-tree with nvcc for sm_100a.

    python -m paper_1908_00587_b200.build [--force]

The transform kernels are instantiated once per line length in separate translation units
(``csrc/nonlinear_inst.cu`` with ``-DNSC_FFT_N=<n>``) so that the build runs in parallel.
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libnsc.so")
FFT_LENGTHS = (12, 24, 48, 96, 192)          # generic kernels; 384, 768, 1536: warp-transform kernels (nonlinear_v2.cu)
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: libnsc.so cannot be built")
    return exe


def _sources():
    units = [("plan", "plan.cu", []), ("api", "api.cu", []), ("linear", "linear.cu", []),
             ("nonlinear", "nonlinear.cu", []), ("nonlinear_v2", "nonlinear_v2.cu", []),
             ("peaks", "peaks.cu", []), ("regrid", "regrid.cu", []),
             ("probe_static", "probe_static.cu", [])]
    units += [(f"nonlinear_inst_{n}", "nonlinear_inst.cu", [f"-DNSC_FFT_N={n}"]) for n in FFT_LENGTHS]
    return units


def _newest_source_mtime() -> float:
    paths = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    paths.append(os.path.join(HERE, "..", "include", "nsc.h"))
    paths.append(os.path.abspath(__file__))
    return max(os.path.getmtime(p) for p in paths)


def _compile(unit):
    name, src, defs = unit
    obj = os.path.join(OBJ, name + ".o")
    cmd = [_nvcc(), *NVCC_FLAGS, *defs, "-c", os.path.join(CSRC, src), "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    with open(os.path.join(OBJ, name + ".log"), "w") as fh:
        fh.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed for {name}:\n{r.stdout}\n{r.stderr}")
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    """Compiles and links libnsc.so unless it is newer than every source; returns its path."""
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest_source_mtime():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    units = _sources()
    with cf.ThreadPoolExecutor(max_workers=min(len(units), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(_compile, units))
    cmd = [_nvcc(), "-shared", "-o", LIB, *objs, "-lcudart"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    if verbose:
        print("built", LIB)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
