"""In-tree build of libem.so for sm_100a (nvcc cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libem.so")
LIB_FUZZ = os.path.join(HERE, "libem_fuzz.so")
SOURCES = ["em_lib.cu"]
HEADERS = ["em_ptx.cuh", "em_common.cuh", "em_split.cuh", "em_aux.cuh", "em_tile.cuh", "em_sweep.cuh", "em_sweep_phaseb.inc", "em_sweep_phaseb_hom.inc", "em_thermal.cuh", os.path.join("..", "..", "include", "em.h")]



def have_nvcc() -> bool:
    return os.path.exists(os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc"))


def _stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build_lib(force: bool = False, verbose: bool = False, fuzz: bool = False, defines=()) -> str:
    """libem.so; fuzz=True builds libem_fuzz.so, the TEST variant with random delays at every synchronisation point of
    the sweep (csrc/em_sweep.cuh "schedule fuzzing") and the extra entry em_fuzz_seed.  defines: extra -D switches for
    the experiment knobs of the sweep (profiles/r2_experiments.md); such a build is always forced and the next plain
    build (any source newer, or --force) replaces it."""
    lib = LIB_FUZZ if fuzz else LIB
    if force or defines or _stale(lib):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
               "-Xcompiler", "-fPIC", "-shared", "-o", lib] + [os.path.join(CSRC, s) for s in SOURCES]
        if fuzz:
            cmd += ["-DEM_SWEEP_FUZZ"]
        cmd += list(defines)
        if verbose:
            cmd += ["-Xptxas", "-v"]
        subprocess.check_call(cmd)
    return lib


if __name__ == "__main__":
    print(build_lib(force="--force" in sys.argv, verbose="-v" in sys.argv, fuzz="--fuzz" in sys.argv,
                    defines=[a for a in sys.argv[1:] if a.startswith("-D")]))
