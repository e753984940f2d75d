"""Build the CUDA library in-tree for sm_100a (nvcc cross-compiles without a GPU).

Two shared objects come out of the same sources:
  libforge_b200.so       the product library: only the instantiations the dispatch tables reach, reads no
                         environment variable (no ablation / grid / variant switches exist in it)
  libforge_b200_prof.so  -DFORGE_PROFILING: the tuning sweeps (FORGE_CFG), grid override (FORGE_GRID) and ablation
                         switches (FORGE_ABLATE) the commands quoted under profiles/ and two tests use
"""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB_PATH = os.path.join(_HERE, "libforge_b200.so")
PROF_LIB_PATH = os.path.join(_HERE, "libforge_b200_prof.so")
SOURCES = ["forge_api.cu"]
HEADERS = ["fused_kernel.cuh", "dgrad_kernel.cuh", "elementwise_kernel.cuh", "adamw_math.cuh", "family_math.cuh", "ptx.cuh",
           "profiling_variants.inc"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--compiler-options", "-fPIC", "-shared"]


def _stale(path: str) -> bool:
    if not os.path.exists(path):
        return True
    t = os.path.getmtime(path)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS]
    deps.append(os.path.join(os.path.dirname(_HERE), "include", "forge.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def _cmd(path: str, profiling: bool, verbose: bool):
    nvcc = os.environ.get("NVCC", "nvcc")
    return [nvcc] + NVCC_FLAGS + (["-DFORGE_PROFILING"] if profiling else []) + (["-Xptxas", "-v"] if verbose else []) + \
           ["-o", path] + [os.path.join(CSRC, s) for s in SOURCES]


def build(force: bool = False, verbose: bool = False, profiling: bool = False) -> str:
    """Compile csrc/*.cu into libforge_b200.so (or, profiling=True, libforge_b200_prof.so); returns its path."""
    path = PROF_LIB_PATH if profiling else LIB_PATH
    if force or _stale(path):
        subprocess.run(_cmd(path, profiling, verbose), check=True)
    return path


def build_all(force: bool = False) -> None:
    """Both libraries, compiled side by side."""
    procs = []
    for profiling in (False, True):
        path = PROF_LIB_PATH if profiling else LIB_PATH
        if force or _stale(path):
            procs.append(subprocess.Popen(_cmd(path, profiling, False)))
    for p in procs:
        if p.wait() != 0:
            raise subprocess.CalledProcessError(p.returncode, p.args)


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose=True, profiling="--profiling" in sys.argv))
