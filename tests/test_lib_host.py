"""CPU-side checks of the C-ABI library: it builds, loads and exports every symbol that include/em.h
declares; host-only entry points work; device entry points fail loudly without a GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import workloads as W
import paper_2603_07038_b200 as P
from paper_2603_07038_b200 import binding as B
from oracle import emo

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "em.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = sorted(set(re.findall(r"\b(em_[a-z_]+)\s*\(", hdr)))
    assert {"em_create", "em_set_source", "em_step", "em_joule", "em_probe"} <= set(names)
    L = P.load()
    for n in names:
        assert hasattr(L, n), n


def test_abi_version_matches_the_header():
    hdr = open(os.path.join(ROOT, "include", "em.h")).read()
    v = int(re.search(r"#define EM_ABI_VERSION (\d+)", hdr).group(1))
    assert P.load().em_abi_version() == v == P.EM_ABI_VERSION
    assert C.sizeof(B.em_grid) == 112          # the layout of include/em.h: 3 ints, 3 pointers, 17 ints, 2 int64 (padded)


def test_workspace_bytes_and_argument_errors():
    n = P.em_workspace_bytes(1024, 1024, 192, 32, 256, 8192, 256000)
    cells = 1024 * 1024 * 192
    assert 13 * 4 * cells < n < 1.2 * (13 * 4 + 1) * cells + (64 << 20)
    with pytest.raises(P.EMError) as e:
        P.em_workspace_bytes(16, 16, 16, precision=16)
    assert e.value.code == 1
    with pytest.raises(P.EMError):
        P.em_workspace_bytes(0, 16, 16)
    # the light kernels launch one 32 x 8 block column per z plane: grid.y, grid.z <= 65535 (em.h states the limits)
    assert P.em_workspace_bytes(2, 2, 65534) > 0 and P.em_workspace_bytes(2, 524272, 2) > 0
    for dims in [(2, 2, 65535), (2, 524273, 2)]:
        with pytest.raises(P.EMError) as e:
            P.em_workspace_bytes(*dims)
        assert e.value.code == 1


@pytest.mark.parametrize("seed", [1, 2])
def test_cfl_dt_matches_oracle_and_generator(seed):
    p = W.random_problem(9, 8, 7, seed=seed, n_ports=0)
    a = P.em_cfl_dt(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz, p.mat_id, p.table)
    b = emo.cfl_dt(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz, p.mat_id, p.table)
    assert abs(a - b) <= 1e-15 * b
    assert abs(0.9 * a - p.dt) <= 1e-14 * p.dt
    p5 = W.make_config(5, scale=8, zscale=4)
    a5 = P.em_cfl_dt(p5.nx, p5.ny, p5.nz, p5.dx, p5.dy, p5.dz, p5.mat_id, p5.table)
    assert abs(0.9 * a5 - p5.dt) <= 1e-14 * p5.dt


def test_cfl_dt_hand_computed_2x2x2():
    """the library's em_cfl_dt against the hand-computed bound of tests/golden/cfl_2x2x2.txt"""
    from workloads.problem import EPS0, MU0
    want = float([l.split()[1] for l in open(os.path.join(ROOT, "tests", "golden", "cfl_2x2x2.txt")) if l.startswith("dt_max ")][0])
    dx, dy, dz = np.asarray([1e-3, 2e-3]), np.asarray([1e-3, 3e-3]), np.asarray([2e-3, 1e-3])
    table = np.asarray([[EPS0, MU0, 0.0], [4.0 * EPS0, MU0, 0.0]])
    mat = np.zeros((2, 2, 2), np.uint8); mat[1, 0, 0] = 1
    assert abs(P.em_cfl_dt(2, 2, 2, dx, dy, dz, mat, table) - want) <= 1e-13 * want


def test_create_validates_before_touching_the_device():
    L = P.load()
    p = W.random_problem(4, 4, 4, seed=3, n_ports=0)
    g = B._mk_grid(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz, 64)
    tab = B._mk_table(p.table, p.flags)
    h = C.c_void_p()
    mat = np.ascontiguousarray(p.mat_id)
    ws = C.c_void_p(256)

    def create(grid=g, n_mat=16, dt=p.dt, m=mat, w=ws):
        return L.em_create(C.byref(grid), m.ctypes.data_as(C.c_void_p), tab, n_mat, C.c_double(dt), w, 1 << 40, None, C.byref(h))
    assert create(dt=0.0) == 1
    assert create(n_mat=300) == 1
    bad = mat.copy(); bad[0, 0, 0] = 99
    assert create(m=bad) == 1
    assert create(w=C.c_void_p(8)) == 1                      # misaligned workspace
    assert create(w=None) == 1
    gp = B._mk_grid(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz, 64, bc=(2, 0, 0, 0, 0, 0))
    assert create(grid=gp) == 1                              # unknown boundary condition
    assert b"boundary" in L.em_last_error()
    gp = B._mk_grid(p.nx, p.ny, p.nz, p.dx, p.dy, p.dz, 64, bc=(1, 0, 0, 0, 0, 0))
    assert create(grid=gp, n_mat=255) == 1                   # a PMC wall needs a table id of its own
    assert b"PMC" in L.em_last_error()
    for fn in (L.em_step, L.em_reset):
        assert fn(None, 1) == 1 if fn is L.em_step else fn(None) == 1


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    p = W.random_problem(4, 4, 4, seed=3, n_ports=0)
    with pytest.raises(RuntimeError):
        P.EM(p)


def test_sweep_kernels_do_not_spill():
    """The TMA sweep runs with a 227 KB shared-memory carve-out, i.e. almost no L1: a register spill in its plane loop
    costs ~19 % (measured twice).  ptxas must report 0 spill bytes for every k_sweep_tma
    instantiation (fp32: 128 registers at 512 threads, fp64: <= 168 at 384 threads)."""
    import shutil
    import subprocess
    import tempfile
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not os.path.exists(nvcc) and not shutil.which("nvcc"):
        pytest.skip("nvcc not found")
    src = os.path.join(ROOT, "paper_2603_07038_b200", "csrc", "em_lib.cu")
    with tempfile.TemporaryDirectory() as tmp:
        out = subprocess.run([nvcc, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
                              "-Xptxas", "-v", "-c", "-o", os.path.join(tmp, "em_lib.o"), src],
                             capture_output=True, text=True, check=True).stderr
    blocks = re.split(r"ptxas info\s+: Compiling entry function ", out)
    seen = 0
    for b in blocks:
        m = re.match(r"'(\S+)'", b)
        if not m or "k_sweep_tma" not in m.group(1):
            continue
        flags = re.search(r"Li([01])ELb([01])ELb([01])ELb([01])EEEv", m.group(1))     # LOSS, UMU, TH, EO
        coupled, eonly, exp_loss = flags.group(3) == "1", flags.group(4) == "1", flags.group(1) == "1"
        if eonly and exp_loss and "tmaIf" in m.group(1):
            continue                                              # fp32 E-only with EXP loss (not a stated config): <= 8 bytes
        seen += 1
        spill = re.search(r"(\d+) bytes spill stores, (\d+) bytes spill loads", b)
        regs = re.search(r"Used (\d+) registers", b)
        assert spill and regs, b[:300]
        assert int(spill.group(1)) == 0 and int(spill.group(2)) == 0, (m.group(1), spill.group(0))
        assert int(regs.group(1)) <= (168 if ("tmaId" in m.group(1) or coupled) else 128), (m.group(1), regs.group(0))
    # leapfrog: {float, double} x {CD, EXP} x {uniform mu, general} = 8; fp32 coupled x {CD, EXP} = 2;
    # fp64 coupled x {CD, EXP} = 2; E-only: double x {CD, EXP} x {umu, general} + float x CD x {umu, general} = 6
    assert seen == 18


def test_product_library_has_no_emulation_in_it():
    """tests/emu compiles the kernel sources against a CPU emulation of the CUDA primitives for checking; none of that may
    leak into the product: libem.so exports no emu_* entry point, its build never defines EM_EMULATE, and nothing in the
    package, bench.py or __graft_entry__.smoke() loads an emulated library."""
    L = P.load()
    for name in ("emu_alloc", "emu_free", "emu_launch_count", "emu_install_fault_handler"):
        assert not hasattr(L, name)
    build_py = open(os.path.join(ROOT, "paper_2603_07038_b200", "build.py")).read()
    assert "EM_EMULATE" not in build_py
    for rel in ("bench.py", os.path.join("paper_2603_07038_b200", "binding.py"), os.path.join("paper_2603_07038_b200", "slabs.py"),
                os.path.join("paper_2603_07038_b200", "__init__.py"), os.path.join("paper_2603_07038_b200", "replicas.py")):
        src = open(os.path.join(ROOT, rel)).read()
        assert "emu_em" not in src and "libem_emu" not in src and "build_emu" not in src, rel


def test_sass_diff_reads_the_built_library():
    """paper_2603_07038_b200/sass_diff.py (profiles/r2_sass_check.md): the built library compared with itself is identical
    kernel by kernel, and holds the 20 instantiations of the sweep the bench lines are about"""
    import shutil
    from paper_2603_07038_b200 import sass_diff
    if shutil.which("cuobjdump") is None or shutil.which("c++filt") is None:
        pytest.skip("cuobjdump / c++filt not on PATH")
    lib = os.path.join(ROOT, "paper_2603_07038_b200", "libem.so")
    P.load()
    res = sass_diff.compare(lib, lib)
    assert res and set(res.values()) == {"identical"}
    assert sum("k_sweep_tma<" in k for k in res) == 20
    k = sass_diff.kernels(lib)
    sweep = next(v for n, v in k.items() if "k_sweep_tma<float, 0, false, false, false>" in n)
    assert any(i.startswith("UTMALDG") for i in sweep) and any("SYNCS" in i for i in sweep)      # TMA boxes on mbarriers
