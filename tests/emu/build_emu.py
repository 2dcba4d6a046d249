"""TEST INFRASTRUCTURE: builds tests/emu/libem_emu*.so -- the product sources paper_2603_07038_b200/csrc/em_lib.cu and
its headers, unmodified, compiled by g++ with -DEM_EMULATE against the CPU emulation of the CUDA primitives in this
folder (emu_cuda.h, em_ptx_emu.h).  The package never loads these libraries; only tests do."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
CSRC = os.path.join(ROOT, "paper_2603_07038_b200", "csrc")


def lib_path(tag: str = "") -> str:
    return os.path.join(HERE, "libem_emu%s.so" % (("_" + tag) if tag else ""))


def _stale(lib: str) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    deps += [os.path.join(HERE, f) for f in ("emu_cuda.h", "em_ptx_emu.h", "emu_exports.cpp", "build_emu.py")]
    deps += [os.path.join(ROOT, "include", "em.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build_emu(tag: str = "", defines=(), force: bool = False, opt: str = "-O2", csrc_dir: str = None, out_dir: str = None) -> str:
    """tag names the variant (libem_emu_<tag>.so); defines: extra -D switches of the kernels, e.g.
    -DEM_SWEEP_FUSED_CONDUCTION=1, or -fsanitize=thread for the racecheck build.  csrc_dir / out_dir: build a (mutated) COPY
    of the kernel sources somewhere else (tests/test_emu_mutations.py)."""
    lib = lib_path(tag) if out_dir is None else os.path.join(out_dir, os.path.basename(lib_path(tag)))
    CSRC = csrc_dir or globals()["CSRC"]
    if force or csrc_dir is not None or _stale(lib):
        cxx = [os.environ.get("CXX", "g++"), opt, "-g", "-std=c++17", "-fPIC", "-pthread", "-DEM_EMULATE",
               "-fno-strict-aliasing", "-Wno-attributes", "-I", os.path.join(HERE, "include"), "-I", HERE, "-I", CSRC]
        obj_lib, obj_exp = lib[:-3] + "_em_lib.o", lib[:-3] + "_exports.o"
        # (the emulation's own runtime file is never instrumented: it IMPLEMENTS the -fsanitize=thread hooks)
        subprocess.check_call(cxx + list(defines) + ["-x", "c++", "-c", os.path.join(CSRC, "em_lib.cu"), "-o", obj_lib])
        subprocess.check_call(cxx + [d for d in defines if not d.startswith("-fsanitize")] +
                              ["-c", os.path.join(HERE, "emu_exports.cpp"), "-o", obj_exp])
        subprocess.check_call(cxx + ["-shared", "-o", lib, obj_lib, obj_exp])
    return lib


VARIANTS = {                             # tag -> extra compiler switches (tests/test_emu_sweep.py)
    "": [],
    "fc": ["-DEM_SWEEP_FUSED_CONDUCTION=1"],
    "race": ["-fsanitize=thread"],
    "race_fc": ["-fsanitize=thread", "-DEM_SWEEP_FUSED_CONDUCTION=1"],
}


def build_all() -> None:
    """every variant the default tests load, and the two self-test libraries, side by side (one compiler process each)"""
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=6) as ex:
        jobs = [ex.submit(build_emu, tag, flags) for tag, flags in VARIANTS.items()]
        jobs += [ex.submit(build_selftest, False, False), ex.submit(build_selftest, False, True)]
        for j in jobs:
            j.result()


RACE_FLAGS = ["-fsanitize=thread"]      # the kernels' loads and stores call the emulation's race detector (emu_exports.cpp)


def build_selftest(force: bool = False, race: bool = False) -> str:
    """tests/emu/libemu_selftest[_race].so: the emulation checked on small kernels with deliberate bugs (selftest.cpp);
    race=True instruments the kernels' loads and stores for the racecheck cases"""
    lib = os.path.join(HERE, "libemu_selftest%s.so" % ("_race" if race else ""))
    srcs = [os.path.join(HERE, f) for f in ("selftest.cpp", "emu_exports.cpp")]
    deps = srcs + [os.path.join(HERE, f) for f in ("emu_cuda.h", "em_ptx_emu.h", "build_emu.py")]
    if force or not os.path.exists(lib) or any(os.path.getmtime(d) > os.path.getmtime(lib) for d in deps):
        cxx = [os.environ.get("CXX", "g++"), "-O1", "-g", "-std=c++17", "-fPIC", "-pthread", "-Wno-attributes",
               "-I", os.path.join(HERE, "include"), "-I", HERE]
        objs = []
        for src, extra in ((srcs[0], RACE_FLAGS if race else []), (srcs[1], [])):
            obj = lib[:-3] + "_" + os.path.basename(src) + ".o"
            subprocess.check_call(cxx + extra + ["-c", src, "-o", obj])
            objs.append(obj)
        subprocess.check_call(cxx + ["-shared", "-o", lib] + objs)
    return lib


if __name__ == "__main__":
    tag = ""
    for a in sys.argv[1:]:
        if a.startswith("--tag="):
            tag = a[6:]
    print(build_emu(tag, [a for a in sys.argv[1:] if a.startswith("-D")], force="--force" in sys.argv))
