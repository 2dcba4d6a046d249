"""Seeded generators for the five BASELINE.json configurations plus small randomised grids.

All randomness: numpy.random.default_rng(2603070380 + k) for config k, drawn in the fixed order
grid -> layout -> ports -> waveforms -> probes.  ``scale`` shrinks nx, ny (and
for configs 4/5 optionally nz via ``zscale``) so that the oracle finishes in seconds in the tests;
feature coordinates scale with the grid, feature sizes in cells (trace width, bump radius) do not.
"""
from __future__ import annotations

import math
from typing import List, Optional, Tuple

import numpy as np

from .problem import (
    Problem, EPS0, MU0, C0, material_table, cfl_dt, LOSS_CD, LOSS_EXP,
    VAC, SI, SIO2, CU, ORG, UF, PI, EMC, DSI, MAG, field_shapes,
)

SEED0 = 2603070380


# --------------------------------------------------------------------------------------------
# helpers (bookkeeping only)
# --------------------------------------------------------------------------------------------
class _Sources:
    """Accumulates ports / edges / waveform tables into the flat arrays of Problem."""

    def __init__(self):
        self.eb: List[int] = []; self.ee: List[int] = []
        self.amp: List[float] = []; self.wo: List[int] = []; self.wl: List[int] = []
        self.comp: List[int] = []; self.ijk: List[Tuple[int, int, int]] = []; self.w: List[float] = []
        self.wave: List[np.ndarray] = []; self._woff = 0

    def add_wave(self, samples: np.ndarray) -> Tuple[int, int]:
        samples = np.ascontiguousarray(samples, dtype=np.float64)
        off = self._woff
        self.wave.append(samples); self._woff += samples.shape[0]
        return off, samples.shape[0]

    def add_port(self, edges, amplitude: float, wave_off: int, wave_len: int):
        """edges: iterable of (comp, i, j, k, weight)."""
        b = len(self.comp)
        for (c, i, j, k, w) in edges:
            self.comp.append(int(c)); self.ijk.append((int(i), int(j), int(k))); self.w.append(float(w))
        self.eb.append(b); self.ee.append(len(self.comp))
        self.amp.append(float(amplitude)); self.wo.append(int(wave_off)); self.wl.append(int(wave_len))

    def apply(self, p: Problem):
        p.port_edge_begin = np.asarray(self.eb, np.int64)
        p.port_edge_end = np.asarray(self.ee, np.int64)
        p.port_amplitude = np.asarray(self.amp, np.float64)
        p.port_wave_offset = np.asarray(self.wo, np.int64)
        p.port_wave_len = np.asarray(self.wl, np.int64)
        p.edge_comp = np.asarray(self.comp, np.int32)
        p.edge_ijk = np.asarray(self.ijk, np.int32).reshape(-1, 3)
        p.edge_weight = np.asarray(self.w, np.float64)
        p.wave = np.concatenate(self.wave) if self.wave else np.zeros(0, np.float64)


def _half_times(steps: int, dt: float) -> np.ndarray:
    """Sample instants of J: t = (n + 1/2) dt."""
    return (np.arange(steps, dtype=np.float64) + 0.5) * dt


def _disc_cells(cx: float, cy: float, r: float, nx: int, ny: int):
    """Cells (i, j) whose centre lies within r of (cx, cy)."""
    i0 = max(0, int(math.floor(cx - r - 1))); i1 = min(nx, int(math.ceil(cx + r + 1)))
    j0 = max(0, int(math.floor(cy - r - 1))); j1 = min(ny, int(math.ceil(cy + r + 1)))
    out = []
    for j in range(j0, j1):
        for i in range(i0, i1):
            if (i + 0.5 - cx) ** 2 + (j + 0.5 - cy) ** 2 <= r * r:
                out.append((i, j))
    return out


def _paint_cylinder(mat, cx, cy, r, k0, k1, mid):
    nz, ny, nx = mat.shape
    cells = _disc_cells(cx, cy, r, nx, ny)
    for (i, j) in cells:
        mat[k0:k1, j, i] = mid
    return cells


def _bump_port_edges(cx, cy, r, k, nx, ny):
    """Ez(., ., k) edges at nodes within r-1 of the bump axis (gap port on top of a bump)."""
    rr = max(r - 1.0, 0.75)
    out = []
    for j in range(max(1, int(math.floor(cy - rr))), min(ny - 1, int(math.ceil(cy + rr))) + 1):
        for i in range(max(1, int(math.floor(cx - rr))), min(nx - 1, int(math.ceil(cx + rr))) + 1):
            if (i - cx) ** 2 + (j - cy) ** 2 <= rr * rr:
                out.append((2, i, j, k, 1.0))
    return out


def _probes_default(p: Problem, rng, n: int = 8):
    shapes = field_shapes(p.nx, p.ny, p.nz)
    pr = []
    for _ in range(n):
        c = int(rng.integers(0, 6)); sz, sy, sx = shapes[c]
        pr.append((c, int(rng.integers(0, sx)), int(rng.integers(0, sy)), int(rng.integers(0, sz))))
    p.probes = np.asarray(pr, np.int32).reshape(-1, 4)


# --------------------------------------------------------------------------------------------
# config 1: PEC cavity, TE101
# --------------------------------------------------------------------------------------------
def config1_cavity(n: int = 16, h: float = 1.0e-3, steps: int = 1000, e0: float = 1.0) -> Problem:
    """PEC cavity n^3 cells, vacuum, initialised with the *sampled* TE101 mode.

    The initial state (E^0, H^{-1/2}) is the input recipe of SURVEY.md 8(c) P1: the sampled
    sinusoid with the numerical angular frequency, so that the staggered pair is one pure mode.
    """
    nx = ny = nz = n
    d = np.full(n, h)
    mat = np.zeros((nz, ny, nx), np.uint8)
    table = material_table(16)
    dt = 0.9 * h / (C0 * math.sqrt(3.0))
    p = Problem("cfg1_cavity", nx, ny, nz, d.copy(), d.copy(), d.copy(), mat, table,
                np.zeros(16, np.int32), dt, LOSS_CD, 64, steps)
    s = math.sin(math.pi / (2 * n))
    wt = (2.0 / dt) * math.asin(C0 * dt * math.sqrt(2.0 * s * s / (h * h)))   # numerical omega
    a_h = e0 * (dt / (MU0 * h)) * s / math.sin(wt * dt / 2.0)
    ph = math.sin(-wt * dt / 2.0)
    shp = field_shapes(nx, ny, nz)
    ii = np.arange(n + 1, dtype=np.float64); ic = np.arange(n, dtype=np.float64) + 0.5
    ey = np.zeros(shp[1]); hx = np.zeros(shp[3]); hz = np.zeros(shp[5])
    # Ey(i,j,k) = E0 sin(pi i/N) sin(pi k/N)
    ey[:, :, :] = e0 * np.sin(math.pi * ii / n)[None, None, :] * np.sin(math.pi * ii / n)[:, None, None]
    # Hx(i,j,k) = A sin(pi i/N) cos(pi (k+1/2)/N) sin(-w dt/2)
    hx[:, :, :] = a_h * ph * np.sin(math.pi * ii / n)[None, None, :] * np.cos(math.pi * ic / n)[:, None, None]
    # Hz(i,j,k) = -A cos(pi (i+1/2)/N) sin(pi k/N) sin(-w dt/2)
    hz[:, :, :] = -a_h * ph * np.cos(math.pi * ic / n)[None, None, :] * np.sin(math.pi * ii / n)[:, None, None]
    p.init = {1: ey, 3: hx, 5: hz}
    p.probes = np.asarray([(1, n // 2, 3, n // 2)], np.int32)
    p.notes = "TE101 sampled mode; omega_num=%r" % wt
    return p


# --------------------------------------------------------------------------------------------
# config 2: layered slab with copper traces, EXP loss, one gap port
# --------------------------------------------------------------------------------------------
def config2_slab(scale: int = 1, steps: Optional[int] = None) -> Problem:
    rng = np.random.default_rng(SEED0 + 2)
    nx, ny, nz = 128 // scale, 128 // scale, 64
    dx = np.full(nx, 2.0e-6); dy = np.full(ny, 2.0e-6); dz = np.full(nz, 1.0e-6)
    mat = np.empty((nz, ny, nx), np.uint8)
    mat[0:16] = SI; mat[16:56] = SIO2; mat[56:64] = VAC
    # 8 traces, 2 cells wide, non-overlapping (min gap 4 cells), 4 per metal layer
    lo, hi = 4, nx - 6
    n_tr = 8 if nx >= 96 else max(2, (nx - 8) // 12 * 2)
    xs: List[int] = []
    tries = 0
    while len(xs) < n_tr:
        x = int(rng.integers(lo, hi))
        tries += 1
        if all(abs(x - y) >= 6 for y in xs):
            xs.append(x)
        elif tries > 200:                 # small scaled grids: rejection got stuck, start over
            xs, tries = [], 0
    layers = [28] * (n_tr // 2) + [40] * (n_tr - n_tr // 2)
    for x, k in zip(xs, layers):
        mat[k, 2:ny - 2, x:x + 2] = CU
    table = material_table(16)
    dt = cfl_dt(dx, dy, dz, mat, table, 0.9)
    if steps is None:
        steps = 5000
    p = Problem("cfg2_slab", nx, ny, nz, dx, dy, dz, mat, table, np.zeros(16, np.int32), dt,
                LOSS_EXP, 64, steps)
    # port: 1-cell gap in trace 0 at j = 8; Jy on the 3 x 2 Ey edges across the gap cross-section
    x0, k0, jg = xs[0], layers[0], 8
    mat[k0, jg, x0:x0 + 2] = SIO2
    src = _Sources()
    tau = 20.0e-12
    t = _half_times(steps, dt)
    w = math.sqrt(math.e) * (t / tau) * np.exp(-t * t / (2 * tau * tau))
    off, ln = src.add_wave(w)
    edges = [(1, i, jg, k, 1.0) for k in (k0, k0 + 1) for i in (x0, x0 + 1, x0 + 2)]
    src.add_port(edges, 1.0e10, off, ln)
    src.apply(p)
    _probes_default(p, rng)
    return p


# --------------------------------------------------------------------------------------------
# config 3: interposer with microbump array, 64 bit-pattern ports
# --------------------------------------------------------------------------------------------
def _bit_waveform(rng, steps, dt, bit_period, edge, delay, nbits=32):
    bits = rng.integers(0, 2, size=nbits).astype(np.float64)
    bits[0] = 1.0                                   # first bit high: something to see at literal time
    t = _half_times(steps, dt) - delay
    lev = np.zeros(steps)
    prev = 0.0
    # raised-cosine edge of length `edge` at the start of each bit period
    idx = np.floor(t / bit_period).astype(np.int64)
    for n in range(steps):
        if t[n] < 0:
            lev[n] = 0.0
            continue
        b = idx[n]
        cur = bits[b % nbits]
        prv = bits[(b - 1) % nbits] if b > 0 else 0.0
        tl = t[n] - b * bit_period
        if tl < edge:
            lev[n] = prv + (cur - prv) * 0.5 * (1.0 - math.cos(math.pi * tl / edge))
        else:
            lev[n] = cur
    return lev


def config3_interposer(scale: int = 1, precision: int = 32, steps: Optional[int] = None,
                       kappa: float = 1.0, n_ports: int = 64) -> Problem:
    rng = np.random.default_rng(SEED0 + 3)
    nx, ny, nz = 512 // scale, 512 // scale, 128
    h = 1.0e-6
    dx = np.full(nx, h); dy = np.full(ny, h); dz = np.full(nz, h)
    mat = np.empty((nz, ny, nx), np.uint8)
    mat[0:40] = ORG; mat[40:56] = VAC; mat[56:128] = SI
    pitch = int(rng.integers(20, 41))
    bumps = []
    for cy in range(pitch // 2 + 4, ny - 8, pitch):
        for cx in range(pitch // 2 + 4, nx - 8, pitch):
            jx, jy = rng.integers(-2, 3, size=2)
            r = int(rng.integers(3, 6))
            bx, by = cx + int(jx), cy + int(jy)
            if bx - r < 2 or by - r < 2 or bx + r > nx - 2 or by + r > ny - 2:
                continue
            _paint_cylinder(mat, float(bx), float(by), float(r), 40, 56, CU)
            bumps.append((bx, by, r))
    table = material_table(16)
    dt = cfl_dt(dx, dy, dz, mat, table, 0.9)
    if steps is None:
        steps = 2000
    p = Problem("cfg3_interposer", nx, ny, nz, dx, dy, dz, mat, table, np.zeros(16, np.int32), dt,
                LOSS_CD, precision, steps)
    n_ports = min(n_ports, len(bumps))
    chosen = rng.choice(len(bumps), size=n_ports, replace=False)
    src = _Sources()
    for b in chosen:
        bx, by, r = bumps[int(b)]
        for (i, j) in _disc_cells(float(bx), float(by), float(r), nx, ny):
            mat[55, j, i] = VAC                                   # gap on top of the bump
        amp = 1.0e9 * (1.0 + 0.2 * float(rng.uniform(-1, 1)))      # PAPER.md L146 amplitude jitter
        delay = float(rng.uniform(0.0, 10.0e-12)) / kappa
        w = _bit_waveform(rng, steps, dt, 50.0e-12 / kappa, 10.0e-12 / kappa, delay)
        off, ln = src.add_wave(w)
        src.add_port(_bump_port_edges(float(bx), float(by), float(r), 55, nx, ny), amp, off, ln)
    src.apply(p)
    _probes_default(p, rng)
    p.notes = "pitch=%d bumps=%d ports=%d kappa=%g" % (pitch, len(bumps), n_ports, kappa)
    return p


# --------------------------------------------------------------------------------------------
# config 4 / 5: full package layout (index-space generator shared by both)
# --------------------------------------------------------------------------------------------
def _package_layout(nx: int, ny: int, nz: int, rng, n_traces: int, n_ports: int):
    """Paints the package of SURVEY.md 8(d) cfg 4 in index space scaled from 1024x1024x192.

    Returns (mat_id, list of port descriptors).  A port descriptor is (family, edges) with
    family 0 = substrate trigger, 1 = logic noise, 2 = HBM data burst.
    """
    fx, fy, fz = nx / 1024.0, ny / 1024.0, nz / 192.0
    X = lambda v: int(round(v * fx)); Y = lambda v: int(round(v * fy)); Z = lambda v: int(round(v * fz))
    mat = np.empty((nz, ny, nx), np.uint8)
    z_sub, z_int, z_rdl, z_uf, z_die, z_top = Z(64), Z(104), Z(112), Z(128), Z(176), nz
    mat[0:z_sub] = ORG; mat[z_sub:z_int] = SI; mat[z_int:z_rdl] = SIO2
    mat[z_rdl:z_uf] = UF; mat[z_uf:z_die] = EMC; mat[z_die:z_top] = VAC
    # logic dies (doped Si) and HBM stacks (repeat of 5 Si + 1 oxide, copper TSVs)
    dies = [(X(x0), Y(y0), X(x0 + 288), Y(y0 + 288)) for x0 in (208, 528) for y0 in (208, 528)]
    for (a, b, c, d) in dies:
        mat[z_uf:z_die, b:d, a:c] = DSI
    hbms = [(X(x0), Y(y0), X(x0 + 128), Y(y0 + 192)) for x0 in (48, 848) for y0 in (112, 416, 720)]
    tsv_pitch = max(8, int(round(24 * min(fx, fy))))
    for (a, b, c, d) in hbms:
        for k in range(z_uf, z_die):
            mat[k, b:d, a:c] = SIO2 if (k - z_uf) % 6 == 5 else SI
        for ty in range(b + tsv_pitch // 2, d - 3, tsv_pitch):
            for tx in range(a + tsv_pitch // 2, c - 3, tsv_pitch):
                ox, oy = rng.integers(-2, 3, size=2)
                x, y = tx + int(ox), ty + int(oy)
                if a + 1 <= x and x + 2 <= c - 1 and b + 1 <= y and y + 2 <= d - 1:
                    mat[z_uf:z_die, y:y + 2, x:x + 2] = CU
    # micro-bumps under every die / HBM footprint through the underfill layer
    bump_pitch = max(12, int(round(32 * min(fx, fy))))
    logic_bumps, hbm_bumps = [], []
    for fam, rects in ((1, dies), (2, hbms)):
        for (a, b, c, d) in rects:
            for cy in range(b + bump_pitch // 2, d - 6, bump_pitch):
                for cx in range(a + bump_pitch // 2, c - 6, bump_pitch):
                    ox, oy = rng.integers(-2, 3, size=2)
                    r = int(rng.integers(3, 6))
                    bx, by = cx + int(ox), cy + int(oy)
                    if bx - r < 2 or by - r < 2 or bx + r > nx - 2 or by + r > ny - 2:
                        continue
                    _paint_cylinder(mat, float(bx), float(by), float(r), z_rdl, z_uf, CU)
                    (logic_bumps if fam == 1 else hbm_bumps).append((bx, by, r))
    # copper traces: 2 wide, 2 thick; 3/4 in the two substrate metal layers, 1/4 in the RDL layer
    m1, m2, m3 = Z(20), Z(44), min(Z(106), z_rdl - 2)
    layer_of = [m1, m2, m3]
    occ = {m1: np.zeros((ny, nx), bool), m2: np.zeros((ny, nx), bool), m3: np.zeros((ny, nx), bool)}
    traces = []
    tries = 0
    lmin, lmax = max(8, X(128)), max(16, X(768))
    while len(traces) < n_traces and tries < 50 * n_traces:
        tries += 1
        kz = layer_of[(0, 1, 0, 1, 0, 1, 2, 2)[len(traces) % 8]]
        horiz = bool(rng.integers(0, 2))
        ln = int(rng.integers(lmin, lmax + 1))
        if horiz:
            ln = min(ln, nx - 8)
            x0 = int(rng.integers(3, nx - ln - 3)); y0 = int(rng.integers(3, ny - 5))
            x1, y1 = x0 + ln, y0 + 2
        else:
            ln = min(ln, ny - 8)
            x0 = int(rng.integers(3, nx - 5)); y0 = int(rng.integers(3, ny - ln - 3))
            x1, y1 = x0 + 2, y0 + ln
        o = occ[kz]
        if o[max(0, y0 - 3):y1 + 3, max(0, x0 - 3):x1 + 3].any():
            continue
        o[y0:y1, x0:x1] = True
        mat[kz:kz + 2, y0:y1, x0:x1] = CU
        traces.append((kz, x0, y0, x1, y1, horiz))
    # ports
    ports = []
    n_sub = max(1, n_ports // 8)
    n_logic = min(len(logic_bumps), n_ports // 2)
    n_hbm = min(len(hbm_bumps), n_ports - n_sub - n_logic)
    sub_traces = [t for t in traces if t[0] in (m1, m2)]
    # substrate: gap port near one end of a trace, J along the trace, alternating polarity in
    # the order of the transverse coordinate ("alternating polarities along y")
    sub_traces = sorted(sub_traces[:n_sub], key=lambda t: (t[2], t[1]))
    for q, (kz, x0, y0, x1, y1, horiz) in enumerate(sub_traces):
        pol = 1.0 if q % 2 == 0 else -1.0
        if horiz:
            ig = x0 + 2
            mat[kz:kz + 2, y0:y1, ig] = ORG
            edges = [(0, ig, j, k, pol) for k in (kz, kz + 1, kz + 2) for j in (y0, y0 + 1, y0 + 2)]
        else:
            jg = y0 + 2
            mat[kz:kz + 2, jg, x0:x1] = ORG
            edges = [(1, i, jg, k, pol) for k in (kz, kz + 1, kz + 2) for i in (x0, x0 + 1, x0 + 2)]
        ports.append((0, edges))
    for fam, lst, cnt in ((1, logic_bumps, n_logic), (2, hbm_bumps, n_hbm)):
        if cnt <= 0:
            continue
        for b in rng.choice(len(lst), size=cnt, replace=False):
            bx, by, r = lst[int(b)]
            kg = z_uf - 1
            for (i, j) in _disc_cells(float(bx), float(by), float(r), nx, ny):
                mat[kg, j, i] = UF
            ports.append((fam, _bump_port_edges(float(bx), float(by), float(r), kg, nx, ny)))
    return mat, ports


def _package_waveforms(p: Problem, ports, rng, steps: int, window_steps: Optional[int] = None):
    """The paper's three waveform families with the 300 ps window mapped onto
    T = window_steps*dt (default: the run length steps*dt), and its deterministic jitter;
    `steps` samples are tabulated."""
    src = _Sources()
    T = (window_steps if window_steps is not None else steps) * p.dt
    u = T / 300.0                                    # "one paper picosecond"
    t = _half_times(steps, p.dt)
    for fam, edges in ports:
        ja = 1.0 + 0.2 * float(rng.uniform(-1, 1))
        jw = 1.0 + 0.1 * float(rng.uniform(-1, 1))
        jp = 10.0 * u * float(rng.uniform(-1, 1))
        if fam == 0:      # Ricker wavelet, t0 = 40 ps, window 20-60 ps
            t0 = 40.0 * u + jp; s = 5.0 * u * jw
            a = ((t - t0) / s) ** 2
            w = (1.0 - a) * np.exp(-0.5 * a)
            amp = 2.0e9
        elif fam == 1:    # continuous 5 GHz sine over 0-300 ps = 1.5 periods over T
            w = np.sin(2.0 * math.pi * 1.5 * (t - jp) / T)
            amp = 5.0e8
        else:             # 40 GHz carrier (12 periods over T) x 3-bit Gaussian pulse train, 80-230 ps
            env = np.zeros_like(t)
            for b in range(3):
                tc = (105.0 + 50.0 * b) * u + jp
                env += np.exp(-0.5 * ((t - tc) / (9.0 * u * jw)) ** 2)
            w = env * np.sin(2.0 * math.pi * 12.0 * (t - jp) / T)
            amp = 1.0e9
        off, ln = src.add_wave(w)
        src.add_port(edges, amp * ja, off, ln)
    src.apply(p)


def config4_package(scale: int = 1, zscale: int = 1, steps: Optional[int] = None,
                    n_ports: int = 256, n_traces: int = 256, precision: int = 32) -> Problem:
    rng = np.random.default_rng(SEED0 + 4)
    nx, ny, nz = 1024 // scale, 1024 // scale, 192 // zscale
    h = 1.0e-6
    dx = np.full(nx, h); dy = np.full(ny, h); dz = np.full(nz, h)
    if scale > 1:
        n_traces = max(8, n_traces // (scale * scale)); n_ports = max(8, n_ports // scale)
    mat, ports = _package_layout(nx, ny, nz, rng, n_traces, n_ports)
    table = material_table(16)
    dt = cfl_dt(dx, dy, dz, mat, table, 0.9)
    if steps is None:
        steps = 1000
    p = Problem("cfg4_package", nx, ny, nz, dx, dy, dz, mat, table, np.zeros(16, np.int32), dt,
                LOSS_CD, precision, steps, joule_every=100)
    _package_waveforms(p, ports, rng, steps)
    _probes_default(p, rng)
    p.notes = "ports=%d" % len(ports)
    return p


def _graded_axis(n: int, centres, w: int, fine=0.5e-6, coarse=50.0e-6, ratio=1.2) -> np.ndarray:
    idx = np.arange(n)
    dist = np.min(np.abs(idx[:, None] - np.asarray(centres)[None, :]), axis=1)
    e = np.maximum(0, dist - w).astype(np.float64)
    return np.minimum(coarse, fine * ratio ** e)


def config5_graded(scale: int = 1, zscale: int = 1, steps: Optional[int] = None,
                   n_ports: int = 256, n_traces: int = 256, precision: int = 32) -> Problem:
    rng = np.random.default_rng(SEED0 + 5)
    nx, ny, nz = 768 // scale, 768 // scale, 256 // zscale
    wxy = max(4, 48 // scale); wz = max(4, 32 // zscale)
    cx = sorted(int(v) for v in rng.integers(nx // 8, nx - nx // 8, size=2))
    cy = sorted(int(v) for v in rng.integers(ny // 8, ny - ny // 8, size=2))
    dx = _graded_axis(nx, cx, wxy); dy = _graded_axis(ny, cy, wxy); dz = _graded_axis(nz, [nz // 2], wz)
    if scale > 1:
        n_traces = max(8, n_traces // (scale * scale)); n_ports = max(8, n_ports // scale)
    mat, ports = _package_layout(nx, ny, nz, rng, n_traces, n_ports)
    table = material_table(16)
    dt = cfl_dt(dx, dy, dz, mat, table, 0.9)
    if steps is None:
        steps = 1000
    p = Problem("cfg5_graded", nx, ny, nz, dx, dy, dz, mat, table, np.zeros(16, np.int32), dt,
                LOSS_CD, precision, steps)
    _package_waveforms(p, ports, rng, steps)
    _probes_default(p, rng)
    p.notes = "centres x=%s y=%s ports=%d" % (cx, cy, len(ports))
    return p


def config6_paper_mesh(scale: int = 1, steps: Optional[int] = None, n_ports: int = 64, n_traces: int = 96,
                       precision: int = 32) -> Problem:
    """NEXT-2 of SURVEY.md 8(f): a run shaped like the paper's own (376 x 408 x 45 cells, EM DOF
    21 088 285, dt = 20 fs, 300 ps = 15 000 steps; L134: ground plane on z = 0; L142: PMC on the rest of the
    EM boundary; L144-L146: Ricker / 5 GHz sine / 40 GHz burst ports with jitter, at PHYSICAL time scale).
    The layout itself (NEC SX-Aurora, Fig. 1) is not public: cfg 4's seeded package generator in index space
    stands in for it, on a non-uniform grid (x, y: 20 um under the dies graded to 60 um; z: 12 um in the
    bump / RDL region graded to 80 um) chosen so that the paper's dt = 20 fs is below 0.9 x the CFL bound."""
    rng = np.random.default_rng(SEED0 + 6)
    nx, ny, nz = 376 // scale, 408 // scale, 45
    dx = _graded_axis(nx, [nx // 2], max(2, nx // 4), fine=20.0e-6, coarse=60.0e-6, ratio=1.05) * scale
    dy = _graded_axis(ny, [ny // 2], max(2, ny // 4), fine=20.0e-6, coarse=60.0e-6, ratio=1.05) * scale
    dz = _graded_axis(nz, [int(round(nz * 116 / 192.0))], 4, fine=12.0e-6, coarse=80.0e-6, ratio=1.2)
    if scale > 1:
        n_traces = max(8, n_traces // scale); n_ports = max(8, n_ports // scale)
    mat, ports = _package_layout(nx, ny, nz, rng, n_traces, n_ports)
    table = material_table(16)
    dt = 20.0e-15
    assert dt <= cfl_dt(dx, dy, dz, mat, table, 0.9), "20 fs must satisfy the CFL rule on this grid"
    if steps is None:
        steps = 15000
    p = Problem("cfg6_paper_mesh", nx, ny, nz, dx, dy, dz, mat, table, np.zeros(16, np.int32), dt,
                LOSS_CD, precision, steps)
    p.bc = (1, 1, 1, 1, 0, 1)                               # PEC ground at z = 0, PMC elsewhere
    _package_waveforms(p, ports, rng, steps, window_steps=15000)
    _probes_default(p, rng)
    p.notes = "ports=%d  Lx=%.2f mm Ly=%.2f mm Lz=%.2f mm" % (len(ports), dx.sum() * 1e3, dy.sum() * 1e3, dz.sum() * 1e3)
    return p


# --------------------------------------------------------------------------------------------
# small randomised heterogeneous / non-uniform grids (parity-only inputs)
# --------------------------------------------------------------------------------------------
def random_problem(nx: int, ny: int, nz: int, seed: int, steps: int = 20, loss_mode: int = LOSS_CD,
                   precision: int = 64, ids=(VAC, SI, SIO2, CU, MAG), uniform: bool = False,
                   n_ports: int = 2, blocky: bool = True, pec_material: bool = False,
                   lossless: bool = False, init_scale: float = 1.0, bc=(0,) * 6) -> Problem:
    """Random ids (blocky or per-cell), random spacings (ratio up to ~3), random initial E and H
    (H scaled by 1/eta0 so both carry comparable energy), a few random single-edge or two-edge
    ports with smooth random waveforms.  bc: wall truncation (-x,+x,-y,+y,-z,+z; 1 = PMC); with a PMC
    wall and n_ports > 0 one extra single-edge port sits ON the first PMC wall (a tangential edge)."""
    rng = np.random.default_rng(seed)
    if uniform:
        dx = np.full(nx, 1.0e-6); dy = np.full(ny, 1.5e-6); dz = np.full(nz, 0.75e-6)
    else:
        dx = 1.0e-6 * rng.uniform(0.5, 1.5, nx); dy = 1.0e-6 * rng.uniform(0.5, 1.5, ny)
        dz = 1.0e-6 * rng.uniform(0.5, 1.5, nz)
    ids = np.asarray(ids, np.uint8)
    if blocky:
        bx, by, bz = max(1, nx // 3), max(1, ny // 3), max(1, nz // 3)
        coarse = rng.integers(0, len(ids), size=((nz + bz - 1) // bz, (ny + by - 1) // by, (nx + bx - 1) // bx))
        mat = ids[np.repeat(np.repeat(np.repeat(coarse, bz, 0), by, 1), bx, 2)[:nz, :ny, :nx]]
        sprinkle = rng.random((nz, ny, nx)) < 0.1
        mat = np.where(sprinkle, ids[rng.integers(0, len(ids), size=(nz, ny, nx))], mat).astype(np.uint8)
    else:
        mat = ids[rng.integers(0, len(ids), size=(nz, ny, nx))].astype(np.uint8)
    mat = np.ascontiguousarray(mat)
    table = material_table(16)
    if lossless:
        table[:, 2] = 0.0
    flags = np.zeros(16, np.int32)
    if pec_material:
        flags[AL_ID] = 1
        mask = rng.random((nz, ny, nx)) < 0.05
        mat[mask] = AL_ID
    dt = cfl_dt(dx, dy, dz, mat, table, 0.9)
    p = Problem("random_%dx%dx%d_s%d" % (nx, ny, nz, seed), nx, ny, nz, dx, dy, dz, mat, table, flags,
                dt, loss_mode, precision, steps)
    shp = field_shapes(nx, ny, nz)
    eta0 = math.sqrt(MU0 / EPS0)
    p.init = {}
    for c in range(6):
        a = rng.standard_normal(shp[c]) * init_scale
        if c >= 3:
            a /= eta0
        p.init[c] = a
    src = _Sources()
    t = _half_times(steps, dt)
    for _ in range(n_ports):
        cands = []
        for _try in range(64):
            c = int(rng.integers(0, 3))
            lim = [nx, ny, nz]
            lo = [1, 1, 1]; hi = [nx - 1, ny - 1, nz - 1]      # node range strictly inside
            lo[c] = 0; hi[c] = lim[c] - 1                      # along the edge: cell index range
            if any(hi[a] < lo[a] for a in range(3)):
                continue
            ijk = [int(rng.integers(lo[a], hi[a] + 1)) for a in range(3)]
            cands = [(c, ijk[0], ijk[1], ijk[2], 1.0)]
            # optional differential partner one node over (weight -1)
            a2 = (c + 1) % 3
            if ijk[a2] + 1 <= hi[a2] and rng.random() < 0.5:
                j2 = list(ijk); j2[a2] += 1
                cands.append((c, j2[0], j2[1], j2[2], -1.0))
            break
        if not cands:
            continue
        if pec_material:
            continue          # keep PEC-material problems source-free (edge fixedness is data dependent)
        f = rng.uniform(0.5, 3.0) / max(steps * dt, 1e-30)
        w = np.sin(2 * math.pi * f * t + rng.uniform(0, 6.28)) * np.exp(-((t - 0.5 * steps * dt) / (0.3 * steps * dt)) ** 2)
        off, ln = src.add_wave(w)
        src.add_port(cands, 1.0e9 * rng.uniform(0.5, 1.5), off, ln)
    pmc = [b for b in range(6) if bc[b]]
    if pmc and n_ports > 0 and not pec_material and min(nx, ny, nz) >= 2:
        b = pmc[0]; a = b // 2                                  # wall normal axis
        c = (a + 1) % 3                                         # a tangential component
        lim = [nx, ny, nz]
        ijk = [0, 0, 0]
        for ax in range(3):
            if ax == a:
                ijk[ax] = 0 if b % 2 == 0 else lim[ax]          # node plane of the wall
            elif ax == c:
                ijk[ax] = int(rng.integers(0, lim[ax]))         # along the edge: cell index
            else:
                ijk[ax] = int(rng.integers(1, max(lim[ax], 2))) # node strictly inside the other axis
        f = rng.uniform(0.5, 3.0) / max(steps * dt, 1e-30)
        w = np.sin(2 * math.pi * f * t + rng.uniform(0, 6.28))
        off, ln = src.add_wave(w)
        src.add_port([(c, ijk[0], ijk[1], ijk[2], 1.0)], 1.0e9 * rng.uniform(0.5, 1.5), off, ln)
    src.apply(p)
    p.bc = tuple(int(v) for v in bc)
    _probes_default(p, rng, 6)
    return p


AL_ID = 14


def impulse_problem() -> Problem:
    """The hand-derivable worked example of SURVEY.md 8(c) P10: 4x4x4 vacuum cells, h = 1 mm,
    dt = 0.9 h/(c0 sqrt 3), one port = the single edge Ez(2,2,1), amplitude 1 A/m^2, wave [1,0,0,..]."""
    n, h = 4, 1.0e-3
    d = np.full(n, h)
    mat = np.zeros((n, n, n), np.uint8)
    table = material_table(16)
    dt = 0.9 * h / (C0 * math.sqrt(3.0))
    p = Problem("impulse_4x4x4", n, n, n, d.copy(), d.copy(), d.copy(), mat, table,
                np.zeros(16, np.int32), dt, LOSS_CD, 64, 3)
    src = _Sources()
    off, ln = src.add_wave(np.asarray([1.0, 0.0, 0.0, 0.0]))
    src.add_port([(2, 2, 2, 1, 1.0)], 1.0, off, ln)
    src.apply(p)
    return p


def make_config(k: int, scale: int = 1, **kw) -> Problem:
    if k == 1:
        return config1_cavity(**kw)
    if k == 2:
        return config2_slab(scale=scale, **kw)
    if k == 3:
        return config3_interposer(scale=scale, **kw)
    if k == 4:
        return config4_package(scale=scale, **kw)
    if k == 5:
        return config5_graded(scale=scale, **kw)
    if k == 6:
        return config6_paper_mesh(scale=scale, **kw)
    raise ValueError("config must be 1..6")
