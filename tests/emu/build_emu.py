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


def build_emu(tag: str = "", defines=(), force: bool = False, opt: str = "-O2") -> str:
    """tag names the variant (libem_emu_<tag>.so); defines: extra -D switches of the kernels, e.g.
    -DEM_SWEEP_FUSED_CONDUCTION=1."""
    lib = lib_path(tag)
    if force or _stale(lib):
        cmd = [os.environ.get("CXX", "g++"), opt, "-g", "-std=c++17", "-fPIC", "-shared", "-pthread", "-DEM_EMULATE",
               "-fno-strict-aliasing", "-Wno-attributes",
               "-I", os.path.join(HERE, "include"), "-I", HERE, "-I", CSRC,
               "-o", lib, "-x", "c++", os.path.join(CSRC, "em_lib.cu"), os.path.join(HERE, "emu_exports.cpp")]
        cmd += list(defines)
        subprocess.check_call(cmd)
    return lib


def build_selftest(force: bool = False) -> str:
    """tests/emu/libemu_selftest.so: the emulation checked on small kernels with deliberate bugs (selftest.cpp)"""
    lib = os.path.join(HERE, "libemu_selftest.so")
    srcs = [os.path.join(HERE, f) for f in ("selftest.cpp", "emu_exports.cpp")]
    deps = srcs + [os.path.join(HERE, f) for f in ("emu_cuda.h", "em_ptx_emu.h")]
    if force or not os.path.exists(lib) or any(os.path.getmtime(d) > os.path.getmtime(lib) for d in deps):
        subprocess.check_call([os.environ.get("CXX", "g++"), "-O1", "-g", "-std=c++17", "-fPIC", "-shared", "-pthread",
                               "-Wno-attributes", "-I", os.path.join(HERE, "include"), "-I", HERE, "-o", lib] + srcs)
    return lib


if __name__ == "__main__":
    tag = ""
    for a in sys.argv[1:]:
        if a.startswith("--tag="):
            tag = a[6:]
    print(build_emu(tag, [a for a in sys.argv[1:] if a.startswith("-D")], force="--force" in sys.argv))
