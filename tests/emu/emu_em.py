"""TEST INFRASTRUCTURE: ``EmuEM`` drives tests/emu/libem_emu*.so -- the product's C-ABI sources compiled against the CPU
emulation of the CUDA primitives (emu_cuda.h) -- through the product's own ctypes binding, with the workspace in guarded
host memory instead of a torch CUDA tensor.  Only tests import this; the package itself has no CPU path."""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
if HERE not in sys.path:
    sys.path.insert(0, HERE)

import paper_2603_07038_b200.binding as B          # noqa: E402
from build_emu import build_emu                     # noqa: E402

_libs = {}


def load_emu(tag: str = "", defines=()):
    """the emulated library variant `tag` (built on demand), with the binding's prototypes"""
    if tag not in _libs:
        L = B._open(build_emu(tag, defines))
        L.emu_alloc.restype = C.c_void_p
        L.emu_alloc.argtypes = [C.c_size_t]
        L.emu_free.argtypes = [C.c_void_p, C.c_size_t]
        L.emu_launch_count.restype = C.c_long
        _libs[tag] = L
    return _libs[tag]


class EmuEM(B.EM):
    """binding.EM on the emulated library: same calls, host memory.  Device-tensor arguments become CPU tensors."""

    def __init__(self, p, precision=None, kernel=B.EM_KERNEL_AUTO, bc=None, formulation=B.EM_FORM_LEAPFROG, z_chunks=0,
                 e_prev=None, tag: str = "", defines=(), load_sources=True, load_init=True, max_ports=None,
                 max_source_edges=None, max_wave_samples=None):
        import torch
        self._torch = torch
        self._L = load_emu(tag, defines)
        self.nx, self.ny, self.nz = int(p.nx), int(p.ny), int(p.nz)
        self.precision = int(precision if precision is not None else p.precision)
        self.dtype = torch.float32 if self.precision == 32 else torch.float64
        self.np_dtype = np.float32 if self.precision == 32 else np.float64
        self.shapes = B._shapes(self.nx, self.ny, self.nz)
        self.device = torch.device("cpu")
        self._dx = np.ascontiguousarray(p.dx, np.float64)
        self._dy = np.ascontiguousarray(p.dy, np.float64)
        self._dz = np.ascontiguousarray(p.dz, np.float64)
        n_ports = int(p.port_amplitude.shape[0])
        n_con = int(p.edge_comp.shape[0])
        self._grid = B._mk_grid(self.nx, self.ny, self.nz, self._dx, self._dy, self._dz, self.precision, int(p.loss_mode),
                                kernel, max_ports if max_ports is not None else max(n_ports, 1),
                                max_source_edges if max_source_edges is not None else max(n_con, 1),
                                max_wave_samples if max_wave_samples is not None else max(int(p.wave.shape[0]), 1),
                                tuple(bc) if bc is not None else tuple(getattr(p, "bc", (0,) * 6)),
                                B._thermal_flag(p), formulation, z_chunks)
        self.formulation = int(formulation)
        nbytes = C.c_size_t()
        self._check(self._L.em_workspace_bytes(C.byref(self._grid), C.byref(nbytes)))
        self.workspace_bytes = int(nbytes.value)
        self._ws_ptr = self._L.emu_alloc(self.workspace_bytes)
        assert self._ws_ptr and self._ws_ptr % 256 == 0
        mat = np.ascontiguousarray(p.mat_id, np.uint8)
        tab = B._mk_table(np.asarray(p.table, np.float64), getattr(p, "flags", None))
        self._h = C.c_void_p()
        self._check(self._L.em_create(C.byref(self._grid), mat.ctypes.data_as(C.c_void_p), tab, len(tab),
                                      C.c_double(float(p.dt)), C.c_void_p(self._ws_ptr), self.workspace_bytes, None,
                                      C.byref(self._h)))
        if load_sources and n_ports > 0:
            self.em_set_source(p)
        if load_init and getattr(p, "init", None):
            for comp, arr in p.init.items():
                if self.formulation == B.EM_FORM_LEAPFROG or comp < 3:
                    self.em_set_field(comp, arr)
        if e_prev is not None:
            for comp in range(3):
                self.em_set_field(6 + comp, e_prev[comp])
        if getattr(p, "thermal", None) is not None:
            self.em_set_thermal(p.thermal)

    def _check(self, rc):
        B._check(rc, self._L)

    # the z-slab halo calls: as in binding.EM, the packed message lives in host memory here
    def em_get_halo(self, k_plane: int, k_layer: int, out, stream=None):
        assert out.dtype == self.dtype and out.is_contiguous() and out.numel() >= self.halo_elems
        B._check(self._L.em_get_halo(self._h, int(k_plane), int(k_layer), C.c_void_p(out.data_ptr()), None), self._L)
        return out

    def em_set_halo(self, k_plane: int, k_layer: int, src, stream=None):
        assert src.dtype == self.dtype and src.is_contiguous() and src.numel() >= self.halo_elems
        B._check(self._L.em_set_halo(self._h, int(k_plane), int(k_layer), C.c_void_p(src.data_ptr()), None), self._L)

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._L.em_destroy(self._h)
            self._h = C.c_void_p()
            self._L.emu_free(C.c_void_p(self._ws_ptr), self.workspace_bytes)
            self._ws_ptr = 0
