"""ctypes binding of the CPU oracle (oracle/em_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA package and shares no code with it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "em_oracle.c")
_LIB = os.path.join(_HERE, "libemo.so")


_SRC2 = os.path.join(_HERE, "em_oracle_eonly.c")
_LIB2 = os.path.join(_HERE, "libemo_eonly.so")
# EMO_SANITIZE=1: both oracles built with -fsanitize=address,undefined into separate files (run the CPU pins with
# LD_PRELOAD=$(gcc -print-file-name=libasan.so))
_SAN = os.environ.get("EMO_SANITIZE", "") == "1"
if _SAN:
    _LIB, _LIB2 = _LIB.replace(".so", "_san.so"), _LIB2.replace(".so", "_san.so")


def _gcc(src: str, lib: str, force: bool) -> str:
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(src):
        cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off"]
        if _SAN:
            cmd += ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
        subprocess.check_call(cmd + ["-o", lib, src, "-lm"])
    return lib


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -shared of both oracles (the E/H leapfrog and the literal E-only recurrence of eq. (2));
    rebuilt when a source is newer than its library.  Returns the path of the leapfrog oracle."""
    _gcc(_SRC2, _LIB2, force)
    return _gcc(_SRC, _LIB, force)


class _Grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("dx", C.POINTER(C.c_double)), ("dy", C.POINTER(C.c_double)), ("dz", C.POINTER(C.c_double)),
                ("loss_mode", C.c_int32), ("bc", C.c_int32 * 6)]


class _Material(C.Structure):
    _fields_ = [("eps", C.c_double), ("mu", C.c_double), ("sigma", C.c_double), ("flags", C.c_int32)]


class _Port(C.Structure):
    _fields_ = [("edge_begin", C.c_int64), ("edge_end", C.c_int64), ("amplitude", C.c_double),
                ("wave_offset", C.c_int64), ("wave_len", C.c_int64)]


class _Edge(C.Structure):
    _fields_ = [("comp", C.c_int32), ("i", C.c_int32), ("j", C.c_int32), ("k", C.c_int32),
                ("weight", C.c_double)]


class _ProbePt(C.Structure):
    _fields_ = [("comp", C.c_int32), ("i", C.c_int32), ("j", C.c_int32), ("k", C.c_int32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.emo_step_index.restype = C.c_int64
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _shapes(nx, ny, nz):
    return [(nz + 1, ny + 1, nx), (nz + 1, ny, nx + 1), (nz, ny + 1, nx + 1),
            (nz, ny, nx + 1), (nz, ny + 1, nx), (nz + 1, ny, nx)]


def _mk_grid(nx, ny, nz, dx, dy, dz, loss_mode, bc=(0,) * 6):
    g = _Grid()
    g.nx, g.ny, g.nz = nx, ny, nz
    g.dx, g.dy, g.dz = _dp(dx), _dp(dy), _dp(dz)
    g.loss_mode = loss_mode
    for b in range(6):
        g.bc[b] = int(bc[b])
    return g


def _mk_table(table, flags):
    n = table.shape[0]
    arr = (_Material * n)()
    for m in range(n):
        arr[m].eps, arr[m].mu, arr[m].sigma = float(table[m, 0]), float(table[m, 1]), float(table[m, 2])
        arr[m].flags = int(flags[m]) if flags is not None else 0
    return arr


def cfl_dt(nx, ny, nz, dx, dy, dz, mat_id, table, flags=None) -> float:
    dx = np.ascontiguousarray(dx, np.float64); dy = np.ascontiguousarray(dy, np.float64)
    dz = np.ascontiguousarray(dz, np.float64)
    mat_id = np.ascontiguousarray(mat_id, np.uint8)
    g = _mk_grid(nx, ny, nz, dx, dy, dz, 0)
    tab = _mk_table(table, flags)
    out = C.c_double()
    rc = lib().emo_cfl_dt(C.byref(g), mat_id.ctypes.data_as(C.c_void_p), tab, table.shape[0], C.byref(out))
    if rc:
        raise RuntimeError("emo_cfl_dt rc=%d" % rc)
    return out.value


def set_threads(n: int) -> int:
    return int(lib().emo_set_threads(int(n)))


class Oracle:
    """fp64 CPU oracle instance built from a workloads.Problem-like object."""

    def __init__(self, p, load_sources: bool = True, load_init: bool = True):
        self.nx, self.ny, self.nz = int(p.nx), int(p.ny), int(p.nz)
        self.shapes = _shapes(self.nx, self.ny, self.nz)
        self._dx = np.ascontiguousarray(p.dx, np.float64)
        self._dy = np.ascontiguousarray(p.dy, np.float64)
        self._dz = np.ascontiguousarray(p.dz, np.float64)
        mat = np.ascontiguousarray(p.mat_id, np.uint8)
        assert mat.shape == (self.nz, self.ny, self.nx)
        g = _mk_grid(self.nx, self.ny, self.nz, self._dx, self._dy, self._dz, int(p.loss_mode),
                     tuple(getattr(p, "bc", (0,) * 6)))
        tab = _mk_table(p.table, p.flags)
        self._h = C.c_void_p()
        rc = lib().emo_create(C.byref(g), mat.ctypes.data_as(C.c_void_p), tab, p.table.shape[0],
                              C.c_double(p.dt), C.byref(self._h))
        if rc:
            raise RuntimeError("emo_create rc=%d" % rc)
        if load_sources and p.n_ports > 0:
            self.set_source(p)
        if load_init and p.init:
            for comp, arr in p.init.items():
                self.set_field(comp, arr)
        self.nodal = False
        if getattr(p, "thermal", None) is not None:
            self.set_thermal(p.thermal, nodal=getattr(p, "thermal_placement", "cell") == "node")

    def close(self):
        if self._h:
            lib().emo_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_source(self, p):
        np_ = p.n_ports
        ports = (_Port * max(np_, 1))()
        for q in range(np_):
            ports[q].edge_begin = int(p.port_edge_begin[q]); ports[q].edge_end = int(p.port_edge_end[q])
            ports[q].amplitude = float(p.port_amplitude[q])
            ports[q].wave_offset = int(p.port_wave_offset[q]); ports[q].wave_len = int(p.port_wave_len[q])
        ne = int(p.edge_comp.shape[0])
        edges = (_Edge * max(ne, 1))()
        for e in range(ne):
            edges[e].comp = int(p.edge_comp[e])
            edges[e].i, edges[e].j, edges[e].k = (int(v) for v in p.edge_ijk[e])
            edges[e].weight = float(p.edge_weight[e])
        wave = np.ascontiguousarray(p.wave, np.float64)
        rc = lib().emo_set_source(self._h, np_, ports, edges, C.c_int64(ne), _dp(wave), C.c_int64(wave.shape[0]))
        if rc:
            raise RuntimeError("emo_set_source rc=%d" % rc)

    def set_field(self, comp: int, arr):
        a = np.ascontiguousarray(arr, np.float64)
        assert a.shape == self.shapes[comp], (a.shape, self.shapes[comp])
        rc = lib().emo_set_field(self._h, comp, _dp(a))
        if rc:
            raise RuntimeError("emo_set_field rc=%d" % rc)

    def get_field(self, comp: int) -> np.ndarray:
        out = np.empty(self.shapes[comp], np.float64)
        rc = lib().emo_get_field(self._h, comp, _dp(out))
        if rc:
            raise RuntimeError("emo_get_field rc=%d" % rc)
        return out

    def fields(self):
        return [self.get_field(c) for c in range(6)]

    def step(self, n: int = 1):
        rc = lib().emo_step(self._h, C.c_int64(n))
        if rc:
            raise RuntimeError("emo_step rc=%d" % rc)

    def joule(self, power: bool = True, energy: bool = True, total: bool = True, reset: bool = False):
        ncell = (self.nz, self.ny, self.nx)
        p = np.empty(ncell, np.float64) if power else None
        q = np.empty(ncell, np.float64) if energy else None
        t = C.c_double()
        rc = lib().emo_joule(self._h, _dp(p) if power else None, _dp(q) if energy else None,
                             C.byref(t) if total else None, int(reset))
        if rc:
            raise RuntimeError("emo_joule rc=%d" % rc)
        return p, q, (t.value if total else None)

    def probe(self, pts) -> np.ndarray:
        pts = np.asarray(pts, np.int32).reshape(-1, 4)
        arr = (_ProbePt * max(len(pts), 1))()
        for n, (c, i, j, k) in enumerate(pts):
            arr[n].comp, arr[n].i, arr[n].j, arr[n].k = int(c), int(i), int(j), int(k)
        out = np.empty(len(pts), np.float64)
        rc = lib().emo_probe(self._h, len(pts), arr, _dp(out))
        if rc:
            raise RuntimeError("emo_probe rc=%d" % rc)
        return out

    def reset(self):
        lib().emo_reset(self._h)

    # ---- thermal coupling (NEXT-1; eq. (4)-(6)) --------------------------------------
    def set_thermal(self, thermal, nodal: bool = False):
        """thermal: (n_mat, 3) float64 rows (rho_cp [J/m^3/K], k [W/m/K], alpha [1/K]); nodal: theta on the mesh nodes
        (the paper's placement, readings N1-N4) instead of per cell (T1-T5)"""
        t = np.ascontiguousarray(thermal, np.float64)
        fn = lib().emo_set_thermal_nodal if nodal else lib().emo_set_thermal
        rc = fn(self._h, _dp(t), int(t.shape[0]))
        if rc:
            raise RuntimeError("emo_set_thermal rc=%d" % rc)
        self.nodal = bool(nodal)

    @property
    def theta_shape(self):
        return (self.nz + 1, self.ny + 1, self.nx + 1) if self.nodal else (self.nz, self.ny, self.nx)

    def temperature_rise(self) -> np.ndarray:
        out = np.empty(self.theta_shape, np.float64)
        rc = lib().emo_get_temperature_rise(self._h, _dp(out))
        if rc:
            raise RuntimeError("emo_get_temperature_rise rc=%d" % rc)
        return out

    def set_temperature_rise(self, theta):
        a = np.ascontiguousarray(theta, np.float64)
        assert a.shape == self.theta_shape
        rc = lib().emo_set_temperature_rise(self._h, _dp(a))
        if rc:
            raise RuntimeError("emo_set_temperature_rise rc=%d" % rc)

    @property
    def step_index(self) -> int:
        return int(lib().emo_step_index(self._h))


# =====================================================================================================================
_lib2 = None


def lib_eonly():
    global _lib2
    if _lib2 is None:
        build()
        _lib2 = C.CDLL(_LIB2)
        _lib2.emo2_step_index.restype = C.c_int64
    return _lib2


class OracleEOnly:
    """fp64 CPU oracle of the paper's literal E-only three-level recurrence, eq. (2)-(3) (oracle/em_oracle_eonly.c;
    NEXT-4 of SURVEY.md 8(f)).  State: e^n (level 0) and e^{n-1} (level 1); p.init entries 0..2 set e^0, entries
    "m0".."m2" (or the argument e_prev) set e^{-1}."""

    def __init__(self, p, load_sources: bool = True, load_init: bool = True, e_prev=None):
        self.nx, self.ny, self.nz = int(p.nx), int(p.ny), int(p.nz)
        self.shapes = _shapes(self.nx, self.ny, self.nz)[:3]
        self._dx = np.ascontiguousarray(p.dx, np.float64)
        self._dy = np.ascontiguousarray(p.dy, np.float64)
        self._dz = np.ascontiguousarray(p.dz, np.float64)
        mat = np.ascontiguousarray(p.mat_id, np.uint8)
        assert mat.shape == (self.nz, self.ny, self.nx)
        g = _mk_grid(self.nx, self.ny, self.nz, self._dx, self._dy, self._dz, int(p.loss_mode),
                     tuple(getattr(p, "bc", (0,) * 6)))
        tab = _mk_table(p.table, p.flags)
        self._h = C.c_void_p()
        rc = lib_eonly().emo2_create(C.byref(g), mat.ctypes.data_as(C.c_void_p), tab, p.table.shape[0],
                                     C.c_double(p.dt), C.byref(self._h))
        if rc:
            raise RuntimeError("emo2_create rc=%d" % rc)
        if load_sources and p.n_ports > 0:
            self.set_source(p)
        if load_init and p.init:
            for comp, arr in p.init.items():
                if comp in (0, 1, 2):
                    self.set_field(0, comp, arr)
        if e_prev is not None:
            for comp in range(3):
                self.set_field(1, comp, e_prev[comp])

    def close(self):
        if self._h:
            lib_eonly().emo2_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_source(self, p):
        np_ = p.n_ports
        ports = (_Port * max(np_, 1))()
        for q in range(np_):
            ports[q].edge_begin = int(p.port_edge_begin[q]); ports[q].edge_end = int(p.port_edge_end[q])
            ports[q].amplitude = float(p.port_amplitude[q])
            ports[q].wave_offset = int(p.port_wave_offset[q]); ports[q].wave_len = int(p.port_wave_len[q])
        ne = int(p.edge_comp.shape[0])
        edges = (_Edge * max(ne, 1))()
        for e in range(ne):
            edges[e].comp = int(p.edge_comp[e])
            edges[e].i, edges[e].j, edges[e].k = (int(v) for v in p.edge_ijk[e])
            edges[e].weight = float(p.edge_weight[e])
        wave = np.ascontiguousarray(p.wave, np.float64)
        rc = lib_eonly().emo2_set_source(self._h, np_, ports, edges, C.c_int64(ne), _dp(wave), C.c_int64(wave.shape[0]))
        if rc:
            raise RuntimeError("emo2_set_source rc=%d" % rc)

    def set_field(self, level: int, comp: int, arr):
        a = np.ascontiguousarray(arr, np.float64)
        assert a.shape == self.shapes[comp], (a.shape, self.shapes[comp])
        rc = lib_eonly().emo2_set_field(self._h, int(level), int(comp), _dp(a))
        if rc:
            raise RuntimeError("emo2_set_field rc=%d" % rc)

    def get_field(self, level: int, comp: int) -> np.ndarray:
        out = np.empty(self.shapes[comp], np.float64)
        rc = lib_eonly().emo2_get_field(self._h, int(level), int(comp), _dp(out))
        if rc:
            raise RuntimeError("emo2_get_field rc=%d" % rc)
        return out

    def fields(self, level: int = 0):
        return [self.get_field(level, c) for c in range(3)]

    def step(self, n: int = 1):
        rc = lib_eonly().emo2_step(self._h, C.c_int64(n))
        if rc:
            raise RuntimeError("emo2_step rc=%d" % rc)

    def joule(self, power: bool = True, energy: bool = True, total: bool = True, reset: bool = False):
        ncell = (self.nz, self.ny, self.nx)
        p = np.empty(ncell, np.float64) if power else None
        q = np.empty(ncell, np.float64) if energy else None
        t = C.c_double()
        rc = lib_eonly().emo2_joule(self._h, _dp(p) if power else None, _dp(q) if energy else None,
                                    C.byref(t) if total else None, int(reset))
        if rc:
            raise RuntimeError("emo2_joule rc=%d" % rc)
        return p, q, (t.value if total else None)

    def probe(self, pts) -> np.ndarray:
        pts = np.asarray(pts, np.int32).reshape(-1, 4)
        arr = (_ProbePt * max(len(pts), 1))()
        for n, (c, i, j, k) in enumerate(pts):
            arr[n].comp, arr[n].i, arr[n].j, arr[n].k = int(c), int(i), int(j), int(k)
        out = np.empty(len(pts), np.float64)
        rc = lib_eonly().emo2_probe(self._h, len(pts), arr, _dp(out))
        if rc:
            raise RuntimeError("emo2_probe rc=%d" % rc)
        return out

    def reset(self):
        lib_eonly().emo2_reset(self._h)

    def set_step_index(self, n: int):
        rc = lib_eonly().emo2_set_step_index(self._h, C.c_int64(int(n)))
        if rc:
            raise RuntimeError("emo2_set_step_index rc=%d" % rc)

    @property
    def step_index(self) -> int:
        return int(lib_eonly().emo2_step_index(self._h))


def set_threads_eonly(n: int) -> int:
    return int(lib_eonly().emo2_set_threads(int(n)))
