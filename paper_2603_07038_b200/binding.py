"""ctypes binding of libem.so -- argument marshalling only; every step runs in the CUDA kernels.

``EM`` wraps one ``em_ctx``: it asks the library for the workspace size, lets PyTorch allocate that
many bytes on the device, and forwards the calls of include/em.h under the same names
(em_set_source, em_set_field, em_get_field, em_step, em_joule, em_probe, em_reset).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

EM_OK = 0
EM_LOSS_CD, EM_LOSS_EXP = 0, 1
EM_KERNEL_AUTO, EM_KERNEL_SPLIT, EM_KERNEL_TMA = 0, 1, 2
EM_FORM_LEAPFROG, EM_FORM_EONLY = 0, 1
EM_ABI_VERSION = 4            # include/em.h: this binding's em_grid layout and signatures

_HERE = os.path.dirname(os.path.abspath(__file__))


class EMError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__("libem error %d: %s" % (code, msg))
        self.code = code


class em_grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("dx", C.POINTER(C.c_double)), ("dy", C.POINTER(C.c_double)), ("dz", C.POINTER(C.c_double)),
                ("precision", C.c_int32), ("loss_mode", C.c_int32), ("bc", C.c_int32 * 6),
                ("kernel", C.c_int32), ("max_ports", C.c_int32),
                ("max_source_edges", C.c_int64), ("max_wave_samples", C.c_int64),
                ("thermal", C.c_int32), ("formulation", C.c_int32), ("z_chunks", C.c_int32), ("pad_", C.c_int32)]


class em_thermal_material(C.Structure):
    _fields_ = [("rho_cp", C.c_double), ("k", C.c_double), ("alpha", C.c_double)]


class em_material(C.Structure):
    _fields_ = [("eps", C.c_double), ("mu", C.c_double), ("sigma", C.c_double),
                ("flags", C.c_int32), ("pad_", C.c_int32)]


class em_port(C.Structure):
    _fields_ = [("edge_begin", C.c_int64), ("edge_end", C.c_int64), ("amplitude", C.c_double),
                ("wave_offset", C.c_int64), ("wave_len", C.c_int64)]


class em_edge(C.Structure):
    _fields_ = [("comp", C.c_int32), ("i", C.c_int32), ("j", C.c_int32), ("k", C.c_int32),
                ("weight", C.c_double)]


class em_probe_pt(C.Structure):
    _fields_ = [("comp", C.c_int32), ("i", C.c_int32), ("j", C.c_int32), ("k", C.c_int32)]


_lib = None


def lib_path() -> str:
    return os.path.join(_HERE, "libem.so")


def load():
    """Load libem.so.  With nvcc at hand the in-tree build runs first (a cheap mtime check: it recompiles only when a
    source or header is newer than the library); without nvcc the built library must be there.  The library's ABI
    version must be this binding's.  Raises otherwise -- there is no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    from .build import build_lib, have_nvcc
    if have_nvcc():
        build_lib()
    elif not os.path.exists(path):
        raise RuntimeError("libem.so is missing and there is no nvcc to build it (python -m paper_2603_07038_b200.build)")
    _lib = _open(path)
    return _lib


def load_fuzz():
    """TEST build of the library with schedule fuzzing in the sweep (build.py fuzz=True; tests/test_gpu_fuzz.py).
    Pass it to EM(..., lib=...); em_fuzz_seed(seed) switches the random delays on (0: off)."""
    from .build import build_lib
    L = _open(build_lib(fuzz=True))
    L.em_fuzz_seed.argtypes = [C.c_uint32]
    return L


def _open(path: str):
    L = C.CDLL(path)
    try:
        abi = int(L.em_abi_version())
    except AttributeError:
        abi = -1
    if abi != EM_ABI_VERSION:
        raise RuntimeError("libem.so has ABI version %d, this binding needs %d: rebuild it "
                           "(python -m paper_2603_07038_b200.build --force)" % (abi, EM_ABI_VERSION))
    L.em_last_error.restype = C.c_char_p
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    L.em_workspace_bytes.argtypes = [C.POINTER(em_grid), C.POINTER(C.c_size_t)]
    L.em_create.argtypes = [C.POINTER(em_grid), vp, C.POINTER(em_material), i32, C.c_double, vp, C.c_size_t, vp, C.POINTER(vp)]
    L.em_destroy.argtypes = [vp]
    L.em_cfl_dt.argtypes = [C.POINTER(em_grid), vp, C.POINTER(em_material), i32, C.POINTER(C.c_double)]
    L.em_set_source.argtypes = [vp, i32, C.POINTER(em_port), C.POINTER(em_edge), i64, C.POINTER(C.c_double), i64]
    L.em_set_field.argtypes = [vp, i32, vp, i32]
    L.em_get_field.argtypes = [vp, i32, vp, i32]
    L.em_get_plane.argtypes = [vp, i32, i32, vp, i32]
    L.em_set_plane.argtypes = [vp, i32, i32, vp, i32]
    L.em_halo_elems.argtypes = [vp, C.POINTER(i64)]
    L.em_get_halo.argtypes = [vp, i32, i32, vp, vp]
    L.em_set_halo.argtypes = [vp, i32, i32, vp, vp]
    L.em_joule_layers.argtypes = [vp, i32, i32, C.POINTER(C.c_double)]
    L.em_wall_offset.argtypes = [vp, i32, i32, i32, C.POINTER(C.c_size_t)]
    L.em_set_peer_halo.argtypes = [vp, i32, i32, C.POINTER(vp)]
    L.em_step.argtypes = [vp, i64]
    L.em_joule.argtypes = [vp, vp, vp, C.POINTER(C.c_double), i32]
    L.em_probe.argtypes = [vp, i32, C.POINTER(em_probe_pt), C.POINTER(C.c_double)]
    L.em_reset.argtypes = [vp]
    L.em_set_thermal.argtypes = [vp, C.POINTER(em_thermal_material), i32]
    L.em_get_temperature_rise.argtypes = [vp, vp, i32]
    L.em_set_temperature_rise.argtypes = [vp, vp, i32]
    L.em_step_index.argtypes = [vp, C.POINTER(i64)]
    L.em_set_step_index.argtypes = [vp, i64]
    L.em_set_joule_energy.argtypes = [vp, vp, i32]
    L.em_check_finite.argtypes = [vp, C.POINTER(i32)]
    L.em_launch_count.argtypes = [vp, C.POINTER(i64)]
    L.em_timing_enable.argtypes = [vp, i32]
    L.em_timing_read.argtypes = [vp, C.POINTER(C.c_char_p), C.POINTER(i64), C.POINTER(C.c_double)]
    return L


def _check(rc: int, L=None):
    """L: the library the call went to (EM(..., lib=...)); default: the product library"""
    if rc != EM_OK:
        raise EMError(rc, (L if L is not None else load()).em_last_error().decode())


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _mk_grid(nx, ny, nz, dx, dy, dz, precision=64, loss_mode=0, kernel=0, max_ports=0,
             max_source_edges=0, max_wave_samples=0, bc=(0,) * 6, thermal=0, formulation=0, z_chunks=0) -> em_grid:
    g = em_grid()
    g.nx, g.ny, g.nz = int(nx), int(ny), int(nz)
    g.dx, g.dy, g.dz = _dp(dx), _dp(dy), _dp(dz)
    g.precision, g.loss_mode, g.kernel = int(precision), int(loss_mode), int(kernel)
    for b in range(6):
        g.bc[b] = int(bc[b])
    g.max_ports, g.max_source_edges, g.max_wave_samples = int(max_ports), int(max_source_edges), int(max_wave_samples)
    g.thermal = int(thermal)
    g.formulation, g.z_chunks = int(formulation), int(z_chunks)
    return g


def _mk_table(table: np.ndarray, flags) -> "C.Array":
    n = table.shape[0]
    arr = (em_material * n)()
    for m in range(n):
        arr[m].eps, arr[m].mu, arr[m].sigma = float(table[m, 0]), float(table[m, 1]), float(table[m, 2])
        arr[m].flags = int(flags[m]) if flags is not None else 0
    return arr


def em_workspace_bytes(nx, ny, nz, precision=64, max_ports=0, max_source_edges=0, max_wave_samples=0) -> int:
    one = np.ones(1)
    g = _mk_grid(nx, ny, nz, one, one, one, precision, 0, 0, max_ports, max_source_edges, max_wave_samples)
    out = C.c_size_t()
    _check(load().em_workspace_bytes(C.byref(g), C.byref(out)))
    return int(out.value)


def em_cfl_dt(nx, ny, nz, dx, dy, dz, mat_id, table, flags=None) -> float:
    dx = np.ascontiguousarray(dx, np.float64); dy = np.ascontiguousarray(dy, np.float64)
    dz = np.ascontiguousarray(dz, np.float64)
    mat_id = np.ascontiguousarray(mat_id, np.uint8)
    g = _mk_grid(nx, ny, nz, dx, dy, dz)
    tab = _mk_table(np.asarray(table, np.float64), flags)
    out = C.c_double()
    _check(load().em_cfl_dt(C.byref(g), mat_id.ctypes.data_as(C.c_void_p), tab, len(tab), C.byref(out)))
    return out.value


def _shapes(nx, ny, nz):
    e = [(nz + 1, ny + 1, nx), (nz + 1, ny, nx + 1), (nz, ny + 1, nx + 1)]
    return e + [(nz, ny, nx + 1), (nz, ny + 1, nx), (nz + 1, ny, nx)] + e     # 6..8: e^{n-1} (E-only contexts)


EM_THERMAL_CELL, EM_THERMAL_NODE = 1, 2


def _thermal_flag(p) -> int:
    """em_grid.thermal of a problem: 0, per cell (p.thermal set), per node (p.thermal_placement == "node")"""
    if getattr(p, "thermal", None) is None:
        return 0
    return EM_THERMAL_NODE if getattr(p, "thermal_placement", "cell") == "node" else EM_THERMAL_CELL


class EM:
    """One em_ctx.  ``p`` is any object with the attributes of workloads.Problem (plain arrays)."""

    def __init__(self, p, precision: Optional[int] = None, kernel: int = EM_KERNEL_AUTO, device="cuda:0",
                 stream=None, bc: Optional[Sequence[int]] = None, load_sources: bool = True, load_init: bool = True,
                 max_ports: Optional[int] = None, max_source_edges: Optional[int] = None,
                 max_wave_samples: Optional[int] = None, formulation: int = EM_FORM_LEAPFROG, z_chunks: int = 0,
                 e_prev=None, lib=None):
        import torch
        self._torch = torch
        self._L = lib if lib is not None else load()
        self.nx, self.ny, self.nz = int(p.nx), int(p.ny), int(p.nz)
        self.precision = int(precision if precision is not None else p.precision)
        self.dtype = torch.float32 if self.precision == 32 else torch.float64
        self.np_dtype = np.float32 if self.precision == 32 else np.float64
        self.shapes = _shapes(self.nx, self.ny, self.nz)
        self.device = torch.device(device)
        if self.device.type != "cuda" or not torch.cuda.is_available():
            raise RuntimeError("paper_2603_07038_b200 needs a CUDA device (there is no CPU fallback)")
        self._dx = np.ascontiguousarray(p.dx, np.float64)
        self._dy = np.ascontiguousarray(p.dy, np.float64)
        self._dz = np.ascontiguousarray(p.dz, np.float64)
        n_ports = int(p.port_amplitude.shape[0])
        n_con = int(p.edge_comp.shape[0])
        self._grid = _mk_grid(self.nx, self.ny, self.nz, self._dx, self._dy, self._dz, self.precision,
                              int(p.loss_mode), kernel,
                              max_ports if max_ports is not None else max(n_ports, 1),
                              max_source_edges if max_source_edges is not None else max(n_con, 1),
                              max_wave_samples if max_wave_samples is not None else max(int(p.wave.shape[0]), 1),
                              tuple(bc) if bc is not None else tuple(getattr(p, "bc", (0,) * 6)),
                              _thermal_flag(p), formulation, z_chunks)
        self.formulation = int(formulation)
        nbytes = C.c_size_t()
        _check(self._L.em_workspace_bytes(C.byref(self._grid), C.byref(nbytes)), self._L)
        self.workspace_bytes = int(nbytes.value)
        with torch.cuda.device(self.device):
            self._ws = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=self.device)
        base = self._ws.data_ptr()
        self._ws_ptr = (base + 255) // 256 * 256
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        mat = np.ascontiguousarray(p.mat_id, np.uint8)
        assert mat.shape == (self.nz, self.ny, self.nx)
        tab = _mk_table(np.asarray(p.table, np.float64), getattr(p, "flags", None))
        self._h = C.c_void_p()
        with torch.cuda.device(self.device):
            _check(self._L.em_create(C.byref(self._grid), mat.ctypes.data_as(C.c_void_p), tab, len(tab),
                                     C.c_double(float(p.dt)), C.c_void_p(self._ws_ptr), self.workspace_bytes,
                                     C.c_void_p(self._stream.cuda_stream), C.byref(self._h)), self._L)
        if load_sources and n_ports > 0:
            self.em_set_source(p)
        if load_init and getattr(p, "init", None):
            for comp, arr in p.init.items():
                if self.formulation == EM_FORM_LEAPFROG or comp < 3:     # (an E-only context has no H)
                    self.em_set_field(comp, arr)
        if e_prev is not None:                                          # E-only: e^{-1}
            for comp in range(3):
                self.em_set_field(6 + comp, e_prev[comp])
        if getattr(p, "thermal", None) is not None:
            self.em_set_thermal(p.thermal)

    # -- lifetime ---------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._torch.cuda.synchronize(self.device)
            self._L.em_destroy(self._h)
            self._h = C.c_void_p()
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- calls of include/em.h ----------------------------------------------------------------
    def em_set_source(self, p):
        n_ports = int(p.port_amplitude.shape[0])
        ports = (em_port * max(n_ports, 1))()
        for q in range(n_ports):
            ports[q].edge_begin = int(p.port_edge_begin[q]); ports[q].edge_end = int(p.port_edge_end[q])
            ports[q].amplitude = float(p.port_amplitude[q])
            ports[q].wave_offset = int(p.port_wave_offset[q]); ports[q].wave_len = int(p.port_wave_len[q])
        ne = int(p.edge_comp.shape[0])
        edges = (em_edge * max(ne, 1))()
        ec = np.asarray(p.edge_comp); ei = np.asarray(p.edge_ijk); ew = np.asarray(p.edge_weight)
        for e in range(ne):
            edges[e].comp = int(ec[e]); edges[e].i = int(ei[e, 0]); edges[e].j = int(ei[e, 1]); edges[e].k = int(ei[e, 2])
            edges[e].weight = float(ew[e])
        wave = np.ascontiguousarray(p.wave, np.float64)
        _check(self._L.em_set_source(self._h, n_ports, ports, edges, ne, _dp(wave), int(wave.shape[0])), self._L)

    def em_set_field(self, comp: int, arr):
        torch = self._torch
        if isinstance(arr, torch.Tensor):
            t = arr.to(device=self.device, dtype=self.dtype).contiguous()
            assert tuple(t.shape) == self.shapes[comp]
            _check(self._L.em_set_field(self._h, comp, C.c_void_p(t.data_ptr()), 1), self._L)
            self._torch.cuda.current_stream(self.device).synchronize()
        else:
            a = np.ascontiguousarray(arr, self.np_dtype)
            assert a.shape == self.shapes[comp], (a.shape, self.shapes[comp])
            _check(self._L.em_set_field(self._h, comp, a.ctypes.data_as(C.c_void_p), 0), self._L)

    def em_get_field(self, comp: int, out=None, device: bool = False):
        """host ndarray by default; device=True returns a torch tensor on the GPU"""
        if device:
            t = out if out is not None else self._torch.empty(self.shapes[comp], dtype=self.dtype, device=self.device)
            _check(self._L.em_get_field(self._h, comp, C.c_void_p(t.data_ptr()), 1), self._L)
            return t
        a = out if out is not None else np.empty(self.shapes[comp], self.np_dtype)
        _check(self._L.em_get_field(self._h, comp, a.ctypes.data_as(C.c_void_p), 0), self._L)
        return a

    def fields(self):
        """leapfrog: Ex, Ey, Ez, Hx, Hy, Hz; E-only: e^n (3 arrays) then e^{n-1} (3 arrays)"""
        comps = range(6) if self.formulation == EM_FORM_LEAPFROG else (0, 1, 2, 6, 7, 8)
        return [self.em_get_field(c) for c in comps]

    def em_get_plane(self, comp: int, k: int, out=None):
        """device tensor [sy][sx] holding plane k of component comp"""
        sh = self.shapes[comp][1:]
        t = out if out is not None else self._torch.empty(sh, dtype=self.dtype, device=self.device)
        _check(self._L.em_get_plane(self._h, comp, int(k), C.c_void_p(t.data_ptr()), 1), self._L)
        return t

    def em_set_plane(self, comp: int, k: int, t):
        assert tuple(t.shape) == tuple(self.shapes[comp][1:]) and t.dtype == self.dtype and t.is_contiguous()
        _check(self._L.em_set_plane(self._h, comp, int(k), C.c_void_p(t.data_ptr()), 1 if t.is_cuda else 0), self._L)

    # z-slab halo (include/em.h): packed [Ex | Ey (| theta)] of one node plane (and the cell layer behind it)
    @property
    def halo_elems(self) -> int:
        n = C.c_int64()
        _check(self._L.em_halo_elems(self._h, C.byref(n)), self._L)
        return int(n.value)

    def em_get_halo(self, k_plane: int, k_layer: int, out, stream=None):
        assert out.is_cuda and out.dtype == self.dtype and out.is_contiguous() and out.numel() >= self.halo_elems
        _check(self._L.em_get_halo(self._h, int(k_plane), int(k_layer), C.c_void_p(out.data_ptr()),
                                   C.c_void_p(stream.cuda_stream) if stream is not None else None), self._L)
        return out

    def em_set_halo(self, k_plane: int, k_layer: int, src, stream=None):
        assert src.is_cuda and src.dtype == self.dtype and src.is_contiguous() and src.numel() >= self.halo_elems
        _check(self._L.em_set_halo(self._h, int(k_plane), int(k_layer), C.c_void_p(src.data_ptr()),
                                   C.c_void_p(stream.cuda_stream) if stream is not None else None), self._L)

    def em_joule_layers(self, k0: int, k1: int) -> float:
        tot = C.c_double()
        _check(self._L.em_joule_layers(self._h, int(k0), int(k1), C.byref(tot)), self._L)
        return tot.value

    def new_halo_buffer(self):
        return self._torch.empty(self.halo_elems, dtype=self.dtype, device=self.device)

    @property
    def workspace_ptr(self) -> int:
        return self._ws_ptr

    def em_wall_offset(self, side: int, parity: int, comp: int) -> int:
        off = C.c_size_t()
        _check(self._L.em_wall_offset(self._h, int(side), int(parity), int(comp), C.byref(off)), self._L)
        return int(off.value)

    def wall_offsets(self, side: int):
        """[parity * 2 + comp] byte offsets of this context's wall plane (what a neighbour needs for em_set_peer_halo)"""
        return [self.em_wall_offset(side, q, c) for q in (0, 1) for c in (0, 1)]

    def em_set_peer_halo(self, side: int, k_send: int, addresses):
        """addresses: four device addresses [parity * 2 + comp] valid in this process, or None to switch the side off"""
        if addresses is None:
            _check(self._L.em_set_peer_halo(self._h, int(side), 0, None), self._L)
            return
        arr = (C.c_void_p * 4)(*[C.c_void_p(int(a)) for a in addresses])
        _check(self._L.em_set_peer_halo(self._h, int(side), int(k_send), arr), self._L)

    # thermal coupling (eq. (4)-(6)); the context must come from a problem with p.thermal set
    def em_set_thermal(self, thermal):
        t = np.ascontiguousarray(thermal, np.float64)
        arr = (em_thermal_material * t.shape[0])()
        for m in range(t.shape[0]):
            arr[m].rho_cp, arr[m].k, arr[m].alpha = float(t[m, 0]), float(t[m, 1]), float(t[m, 2])
        _check(self._L.em_set_thermal(self._h, arr, int(t.shape[0])), self._L)

    @property
    def theta_shape(self):
        return (self.nz + 1, self.ny + 1, self.nx + 1) if self._grid.thermal == EM_THERMAL_NODE else (self.nz, self.ny, self.nx)

    def em_get_temperature_rise(self, out=None, device: bool = False):
        shape = self.theta_shape
        if device:
            t = out if out is not None else self._torch.empty(shape, dtype=self.dtype, device=self.device)
            _check(self._L.em_get_temperature_rise(self._h, C.c_void_p(t.data_ptr()), 1), self._L)
            return t
        a = out if out is not None else np.empty(shape, self.np_dtype)
        _check(self._L.em_get_temperature_rise(self._h, a.ctypes.data_as(C.c_void_p), 0), self._L)
        return a

    def em_set_temperature_rise(self, theta):
        if self._torch.is_tensor(theta):
            t = theta.to(device=self.device, dtype=self.dtype).contiguous()
            _check(self._L.em_set_temperature_rise(self._h, C.c_void_p(t.data_ptr()), 1), self._L)
            return
        a = np.ascontiguousarray(theta, self.np_dtype)
        assert a.shape == self.theta_shape
        _check(self._L.em_set_temperature_rise(self._h, a.ctypes.data_as(C.c_void_p), 0), self._L)

    def em_step(self, n: int = 1):
        _check(self._L.em_step(self._h, int(n)), self._L)

    def em_joule(self, power=None, energy=None, total: bool = False, reset: bool = False):
        """power / energy: torch device tensors (nz, ny, nx) of the working dtype, or None."""
        tot = C.c_double()
        _check(self._L.em_joule(self._h,
                                C.c_void_p(power.data_ptr()) if power is not None else None,
                                C.c_void_p(energy.data_ptr()) if energy is not None else None,
                                C.byref(tot) if total else None, int(reset)), self._L)
        return tot.value if total else None

    def joule_maps(self, reset: bool = False):
        """convenience: (power ndarray, energy ndarray, total float)"""
        torch = self._torch
        pw = torch.empty((self.nz, self.ny, self.nx), dtype=self.dtype, device=self.device)
        q = torch.empty_like(pw)
        tot = self.em_joule(pw, q, total=True, reset=reset)
        return pw.cpu().numpy(), q.cpu().numpy(), tot

    def em_probe(self, pts) -> np.ndarray:
        pts = np.asarray(pts, np.int32).reshape(-1, 4)
        arr = (em_probe_pt * max(len(pts), 1))()
        for n, (c, i, j, k) in enumerate(pts):
            arr[n].comp, arr[n].i, arr[n].j, arr[n].k = int(c), int(i), int(j), int(k)
        out = np.empty(len(pts), np.float64)
        _check(self._L.em_probe(self._h, len(pts), arr, _dp(out)), self._L)
        return out

    # checkpoint / resume and failure detection (include/em.h)
    def em_set_joule_energy(self, q):
        if self._torch.is_tensor(q):
            t = q.to(device=self.device, dtype=self.dtype).contiguous()
            assert tuple(t.shape) == (self.nz, self.ny, self.nx)
            _check(self._L.em_set_joule_energy(self._h, C.c_void_p(t.data_ptr()), 1 if t.is_cuda else 0), self._L)
            return
        a = np.ascontiguousarray(q, self.np_dtype)
        assert a.shape == (self.nz, self.ny, self.nx)
        _check(self._L.em_set_joule_energy(self._h, a.ctypes.data_as(C.c_void_p), 0), self._L)

    def em_set_step_index(self, n: int):
        _check(self._L.em_set_step_index(self._h, int(n)), self._L)

    def em_check_finite(self) -> bool:
        ok = C.c_int32()
        _check(self._L.em_check_finite(self._h, C.byref(ok)), self._L)
        return bool(ok.value)

    def checkpoint(self) -> dict:
        """the whole state of the run as host arrays (include/em.h "checkpoint / resume")"""
        comps = range(6) if self.formulation == EM_FORM_LEAPFROG else (0, 1, 2, 6, 7, 8)
        ck = {"fields": {c: self.em_get_field(c) for c in comps}, "q": self.joule_maps()[1], "step": self.step_index}
        if (self._grid.thermal):
            ck["theta"] = self.em_get_temperature_rise()
        return ck

    def resume(self, ck: dict):
        """restore a checkpoint into a context created with the same grid, materials, dt and sources"""
        for c, f in ck["fields"].items():
            self.em_set_field(c, f)
        self.em_set_joule_energy(ck["q"])
        if "theta" in ck:
            self.em_set_temperature_rise(ck["theta"])
        self.em_set_step_index(ck["step"])

    def em_reset(self):
        _check(self._L.em_reset(self._h), self._L)

    @property
    def step_index(self) -> int:
        n = C.c_int64()
        _check(self._L.em_step_index(self._h, C.byref(n)), self._L)
        return int(n.value)

    @property
    def launch_count(self) -> int:
        n = C.c_int64()
        _check(self._L.em_launch_count(self._h, C.byref(n)), self._L)
        return int(n.value)

    def em_timing_enable(self, enable: bool = True):
        _check(self._L.em_timing_enable(self._h, int(enable)), self._L)

    def em_timing_read(self):
        name = C.c_char_p(); n = C.c_int64(); ms = C.c_double()
        _check(self._L.em_timing_read(self._h, C.byref(name), C.byref(n), C.byref(ms)), self._L)
        return (name.value or b"").decode(), int(n.value), float(ms.value)
