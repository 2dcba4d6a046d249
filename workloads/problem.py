"""Problem container, physical constants and the shared material table (inputs only)."""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, Optional

import numpy as np

# Physical constants (SI).  They live only here: the library and the oracle see absolute
# eps [F/m], mu [H/m], sigma [S/m] (SURVEY.md 8(c) "Grid, unknowns, constants").
C0 = 299792458.0
MU0 = 4.0e-7 * math.pi
EPS0 = 1.0 / (MU0 * C0 * C0)

LOSS_CD = 0   # paper eq. (3): M, K = D_eps +- dt/2 D_sigma
LOSS_EXP = 1  # exponential-loss update (BASELINE.json config 2)
BC_PEC = 0    # tangential E = 0 on the wall (north_star, configs 1-5; ground plane PAPER.md L134)
BC_PMC = 1    # the paper's EM truncation: tangential H = 0 on the wall

# Shared 16-entry table: ids 0-4 from BASELINE.json, 5-15 generator constants (handbook-order
# values, NOT from the paper: PAPER.md L136-L138 prints mechanical constants only).
#            name                 eps_r  mu_r  sigma [S/m]
_MATERIALS = [
    ("vacuum",              1.0,  1.0, 0.0),
    ("silicon",            11.9,  1.0, 10.0),
    ("sio2",                3.9,  1.0, 0.0),
    ("copper",              1.0,  1.0, 5.8e7),
    ("organic_substrate",   3.5,  1.0, 1.0e-3),
    ("underfill",           3.6,  1.0, 0.0),
    ("polyimide",           3.3,  1.0, 0.0),
    ("epoxy_mould",         4.0,  1.0, 1.0e-5),
    ("bt_resin",            4.5,  1.0, 1.0e-4),
    ("solder",              1.0,  1.0, 7.0e6),
    ("lowk_oxide",          2.9,  1.0, 0.0),
    ("sin",                 7.0,  1.0, 0.0),
    ("doped_si",           11.9,  1.0, 100.0),
    ("tsv_liner",           3.9,  1.0, 0.0),
    ("aluminium",           1.0,  1.0, 3.5e7),
    ("test_magnetic",       2.0,  2.0, 0.0),
]
MATERIAL_NAMES = [m[0] for m in _MATERIALS]
VAC, SI, SIO2, CU, ORG, UF, PI, EMC, BT, SOLDER, LOWK, SIN, DSI, LINER, AL, MAG = range(16)


# Thermal constants of the same 16 materials (handbook-order values, NOT from the paper, which prints mechanical
# constants only): rho*c_p [J/m^3/K], k [W/m/K], alpha = temperature coefficient of resistance [1/K]
_THERMAL = [
    (1.2e3,   0.026, 0.0),      # vacuum / air
    (1.63e6, 148.0,  0.0),      # silicon
    (1.61e6,   1.4,  0.0),      # sio2
    (3.45e6, 400.0,  3.9e-3),   # copper
    (1.8e6,    0.3,  0.0),      # organic substrate
    (1.9e6,    0.5,  0.0),      # underfill
    (1.55e6,   0.2,  0.0),      # polyimide
    (1.7e6,    0.8,  0.0),      # epoxy mould
    (1.8e6,    0.35, 0.0),      # BT resin
    (1.67e6,  50.0,  4.0e-3),   # solder
    (1.4e6,    0.6,  0.0),      # low-k oxide
    (2.2e6,   20.0,  0.0),      # SiN
    (1.63e6, 130.0,  0.0),      # doped Si
    (1.61e6,   1.4,  0.0),      # TSV liner
    (2.42e6, 237.0,  4.3e-3),   # aluminium
    (2.0e6,    1.0,  0.0),      # test magnetic
]


def thermal_table(n: int = 16) -> np.ndarray:
    """(n, 3) float64 array of (rho*c_p, k, alpha)."""
    return np.asarray(_THERMAL[:n], np.float64).copy()


def material_table(n: int = 16) -> np.ndarray:
    """(n, 3) float64 array of absolute (eps, mu, sigma)."""
    t = np.empty((n, 3), dtype=np.float64)
    for m in range(n):
        _, er, mr, sg = _MATERIALS[m]
        t[m] = (er * EPS0, mr * MU0, sg)
    return t


@dataclasses.dataclass
class Problem:
    """All inputs of one run, as dense arrays in the logical layout of include/em.h.

    Field shapes (x fastest, C order [k][j][i]):
      Ex (nz+1, ny+1, nx)   Ey (nz+1, ny, nx+1)   Ez (nz, ny+1, nx+1)
      Hx (nz, ny, nx+1)     Hy (nz, ny+1, nx)     Hz (nz+1, ny, nx)
    """
    name: str
    nx: int
    ny: int
    nz: int
    dx: np.ndarray            # (nx,) float64 cell sizes
    dy: np.ndarray
    dz: np.ndarray
    mat_id: np.ndarray        # (nz, ny, nx) uint8
    table: np.ndarray         # (n_mat, 3) float64 eps, mu, sigma (absolute)
    flags: np.ndarray         # (n_mat,) int32, bit0 = PEC material
    dt: float
    loss_mode: int = LOSS_CD
    precision: int = 64       # working precision of the GPU run (the oracle is always fp64)
    steps: int = 0
    # sources: port p drives edges[edge_begin[p]:edge_end[p]] with
    #   J = amplitude[p] * weight[e] * wave[wave_offset[p] + n]   for n < wave_len[p], else 0
    port_edge_begin: np.ndarray = dataclasses.field(default_factory=lambda: np.zeros(0, np.int64))
    port_edge_end: np.ndarray = dataclasses.field(default_factory=lambda: np.zeros(0, np.int64))
    port_amplitude: np.ndarray = dataclasses.field(default_factory=lambda: np.zeros(0, np.float64))
    port_wave_offset: np.ndarray = dataclasses.field(default_factory=lambda: np.zeros(0, np.int64))
    port_wave_len: np.ndarray = dataclasses.field(default_factory=lambda: np.zeros(0, np.int64))
    edge_comp: np.ndarray = dataclasses.field(default_factory=lambda: np.zeros(0, np.int32))
    edge_ijk: np.ndarray = dataclasses.field(default_factory=lambda: np.zeros((0, 3), np.int32))
    edge_weight: np.ndarray = dataclasses.field(default_factory=lambda: np.zeros(0, np.float64))
    wave: np.ndarray = dataclasses.field(default_factory=lambda: np.zeros(0, np.float64))
    probes: np.ndarray = dataclasses.field(default_factory=lambda: np.zeros((0, 4), np.int32))
    init: Optional[Dict[int, np.ndarray]] = None   # comp (0..5 = Ex,Ey,Ez,Hx,Hy,Hz) -> array
    joule_every: int = 0      # config 4: Joule map output every 100 steps
    # wall truncation, order -x, +x, -y, +y, -z, +z: BC_PEC (tangential E = 0) or BC_PMC
    bc: tuple = (0, 0, 0, 0, 0, 0)
    # thermal coupling (eq. (4)-(6)): None = EM only; else (n_mat, 3) float64 rows
    # (rho*c_p [J/m^3/K], k [W/m/K], alpha [1/K]) -> temperature rise per cell and sigma(T) feedback
    thermal: Optional[np.ndarray] = None
    notes: str = ""

    @property
    def n_cells(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def n_ports(self) -> int:
        return int(self.port_amplitude.shape[0])

    def field_shape(self, comp: int):
        nx, ny, nz = self.nx, self.ny, self.nz
        return [
            (nz + 1, ny + 1, nx), (nz + 1, ny, nx + 1), (nz, ny + 1, nx + 1),
            (nz, ny, nx + 1), (nz, ny + 1, nx), (nz + 1, ny, nx),
        ][comp]


def field_shapes(nx: int, ny: int, nz: int):
    return [
        (nz + 1, ny + 1, nx), (nz + 1, ny, nx + 1), (nz, ny + 1, nx + 1),
        (nz, ny, nx + 1), (nz, ny + 1, nx), (nz + 1, ny, nx),
    ]


def cfl_dt(dx, dy, dz, mat_id, table, factor: float = 0.9) -> float:
    """Input recipe for dt ("constrained by the CFL condition"):
    dt = factor * min_c sqrt(eps_c mu_c) / sqrt(dx_i^-2 + dy_j^-2 + dz_k^-2).

    This is a generator-side restatement used only to *choose* the input dt; the library's
    em_cfl_dt and the oracle's emo_cfl_dt implement the same rule independently and are checked
    against each other in the tests.
    """
    dx = np.asarray(dx, np.float64); dy = np.asarray(dy, np.float64); dz = np.asarray(dz, np.float64)
    slow = np.sqrt(table[:, 0] * table[:, 1])            # 1/c per material
    gx = 1.0 / (dx * dx); gy = 1.0 / (dy * dy); gz = 1.0 / (dz * dz)
    best = np.inf
    gxy = gy[:, None] + gx[None, :]
    for k in range(mat_id.shape[0]):
        v = slow[mat_id[k]] / np.sqrt(gxy + gz[k])
        m = float(v.min())
        if m < best:
            best = m
    return factor * best
