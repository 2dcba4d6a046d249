"""Pins of the oracle's PMC walls (the paper's EM truncation; reading C8 of SURVEY.md 8(c):
the wall's tangential E stays an unknown, its dual face is the half face inside, H outside is 0).

None compares the oracle with itself on the same path:
 * mirror image: a PMC wall is the symmetry plane of the domain mirrored in it (tangential E even,
   tangential H odd) -- the half domain with a PMC wall must reproduce the doubled all-PEC domain, whose
   update is pinned by P0-P10 and never touches the PMC code;
 * quarter-wave resonator closed form (PEC at z = 0, PMC at z = L): the sampled mode is an exact discrete
   eigenvector with the numerical resonance w~ = (2/dt) asin(c dt/h sin(pi/4N));
 * discrete energy conservation and Poynting balance with mixed PEC/PMC walls (tests/discrete.py);
 * the dense eq. (2)-(3) brute force with PMC walls is in test_oracle_dense.py.
"""
import copy
import math

import numpy as np
import pytest

import workloads as W
from workloads.problem import LOSS_CD, LOSS_EXP, EPS0, MU0, C0, BC_PEC, BC_PMC, material_table, Problem
from oracle import emo
import discrete as D

AX = {0: 2, 1: 1, 2: 0}          # x, y, z -> numpy axis of the [k][j][i] arrays


def _nodal(comp, a):
    """is component comp (0..2 E, 3..5 H) sampled on node planes along axis a?"""
    return (comp % 3 != a) if comp < 3 else (comp % 3 == a)


def _sign(comp, a):
    """parity under the mirror a -> -a: E polar (normal component flips), H axial (tangential flip)"""
    return (-1.0 if comp == a else 1.0) if comp < 3 else (1.0 if comp - 3 == a else -1.0)


def _mirror_field(arr, comp, a, hi):
    ax = AX[a]
    img = np.flip(arr, ax) * _sign(comp, a)
    if _nodal(comp, a):                     # the wall plane itself is not duplicated
        img = np.delete(img, 0 if hi else -1, ax)
    return np.concatenate([arr, img] if hi else [img, arr], ax)


def _half_of(full, comp, a, hi, n_half):
    ax = AX[a]
    ln = n_half + 1 if _nodal(comp, a) else n_half
    sl = [slice(None)] * 3
    sl[ax] = slice(0, ln) if hi else slice(full.shape[ax] - ln, None)
    return full[tuple(sl)]


def _mirror_problem(p, a, hi):
    """the all-"other-wall" domain obtained by mirroring p in its wall (axis a, hi side)"""
    n = [p.nx, p.ny, p.nz]
    d = [p.dx, p.dy, p.dz]
    d2 = list(d)
    d2[a] = np.concatenate([d[a], d[a][::-1]] if hi else [d[a][::-1], d[a]])
    img = np.flip(p.mat_id, AX[a])
    mat2 = np.ascontiguousarray(np.concatenate([p.mat_id, img] if hi else [img, p.mat_id], AX[a]))
    n2 = list(n); n2[a] = 2 * n[a]
    bc2 = list(p.bc)
    other = p.bc[2 * a + (0 if hi else 1)]
    bc2[2 * a] = bc2[2 * a + 1] = other
    q = Problem(p.name + "_mirrored", n2[0], n2[1], n2[2], d2[0].copy(), d2[1].copy(), d2[2].copy(), mat2,
                p.table, p.flags, p.dt, p.loss_mode, p.precision, p.steps)
    q.bc = tuple(bc2)
    comp, ijk, wt, beg, end = [], [], [], [], []
    for pt in range(p.n_ports):
        beg.append(len(comp))
        for e in range(p.port_edge_begin[pt], p.port_edge_end[pt]):
            c = int(p.edge_comp[e]); idx = [int(v) for v in p.edge_ijk[e]]
            nodal = (c != a)
            orig = list(idx); image = list(idx)
            if hi:
                image[a] = 2 * n[a] - idx[a] if nodal else 2 * n[a] - 1 - idx[a]
            else:
                orig[a] = idx[a] + n[a]
                image[a] = n[a] - idx[a] if nodal else n[a] - 1 - idx[a]
            comp.append(c); ijk.append(orig); wt.append(float(p.edge_weight[e]))
            if image != orig:                         # an edge ON the wall is its own image
                comp.append(c); ijk.append(image); wt.append(float(p.edge_weight[e]) * _sign(c, a))
        end.append(len(comp))
    q.port_edge_begin = np.asarray(beg, np.int64); q.port_edge_end = np.asarray(end, np.int64)
    q.port_amplitude = p.port_amplitude.copy()
    q.port_wave_offset = p.port_wave_offset.copy(); q.port_wave_len = p.port_wave_len.copy()
    q.edge_comp = np.asarray(comp, np.int32); q.edge_ijk = np.asarray(ijk, np.int32).reshape(-1, 3)
    q.edge_weight = np.asarray(wt, np.float64); q.wave = p.wave.copy()
    if p.init is not None:
        q.init = {c: np.ascontiguousarray(_mirror_field(p.init[c], c, a, hi)) for c in p.init}
    return q


@pytest.mark.parametrize("wall", range(6))
@pytest.mark.parametrize("mode", [LOSS_CD, LOSS_EXP])
def test_pmc_wall_equals_mirror_image(wall, mode):
    a, hi = wall // 2, wall % 2 == 1
    bc = [BC_PEC] * 6
    bc[wall] = BC_PMC
    steps = 60
    p = W.random_problem(6, 5, 4, seed=300 + wall, loss_mode=mode, steps=steps, n_ports=2, bc=tuple(bc))
    # the oracle zeroes E on PEC-fixed edges at set_field; zero the same entries of the mirrored input
    for c in range(3):
        p.init[c] = np.where(D.fixed_mask(p.nx, p.ny, p.nz, c, bc=p.bc), 0.0, p.init[c])
    q = _mirror_problem(p, a, hi)
    assert q.bc == (BC_PEC,) * 6
    assert any(int(p.edge_ijk[e][a]) in (0, [p.nx, p.ny, p.nz][a]) and int(p.edge_comp[e]) != a
               for e in range(len(p.edge_comp))), "no port edge on the PMC wall"
    oh, of = emo.Oracle(p), emo.Oracle(q)
    oh.step(steps); of.step(steps)
    fh, ff = oh.fields(), of.fields()
    n_half = [p.nx, p.ny, p.nz][a]
    for grp in ((0, 1, 2), (3, 4, 5)):
        num = sum(np.sum((_half_of(ff[c], c, a, hi, n_half) - fh[c]) ** 2) for c in grp)
        den = sum(np.sum(fh[c] ** 2) for c in grp)
        assert den > 0 and math.sqrt(num / den) < 1e-12, (grp, math.sqrt(num / den))
    # tangential E on the wall is alive (otherwise the test would not exercise the PMC update)
    tang = [c for c in range(3) if c != a]
    sl = [slice(None)] * 3; sl[AX[a]] = -1 if hi else 0
    assert max(np.max(np.abs(fh[c][tuple(sl)])) for c in tang) > 0
    # Joule energy density of the half = that of the matching half of the mirrored domain; totals 1 : 2
    _, qh, Qh = oh.joule(); _, qf, Qf = of.joule()
    sl = [slice(None)] * 3; sl[AX[a]] = slice(0, n_half) if hi else slice(n_half, None)
    assert np.linalg.norm(qf[tuple(sl)] - qh) <= 1e-12 * np.linalg.norm(qh)
    assert Qh > 0 and abs(Qf / Qh - 2.0) < 1e-12


def test_pmc_quarter_wave_closed_form():
    """PEC at z = 0, PMC at z = L = N h (and PMC on the y walls so that Ex may be uniform in y): the
    sampled quarter-wave mode Ex(k) = sin(beta k h), beta = pi/(2 N h), is an exact eigenvector of the
    discrete operator (the mirror image of cos(beta (k+1/2) h) about k = N is its negative), hence
    Ex^n(k) = sin(beta k h) cos(w~ n dt) with w~ = (2/dt) asin(c0 dt/h sin(beta h/2))."""
    N, h, steps = 16, 1.0e-3, 800
    nx, ny = 3, 2
    d = lambda n: np.full(n, h)
    mat = np.zeros((N, ny, nx), np.uint8)
    dt = 0.9 * h / (C0 * math.sqrt(3.0))
    p = Problem("quarter_wave", nx, ny, N, d(nx), d(ny), d(N), mat, material_table(16), np.zeros(16, np.int32),
                dt, LOSS_CD, 64, steps)
    p.bc = (BC_PEC, BC_PEC, BC_PMC, BC_PMC, BC_PEC, BC_PMC)
    beta = math.pi / (2 * N * h)
    wt = 2.0 / dt * math.asin(C0 * dt / h * math.sin(beta * h / 2))
    A = -(dt / (MU0 * h)) * math.sin(beta * h / 2) / math.sin(wt * dt / 2)
    shp = p.field_shape
    k_node = np.arange(N + 1)[:, None, None]; k_cell = (np.arange(N) + 0.5)[:, None, None]
    p.init = {c: np.zeros(shp(c)) for c in range(6)}
    p.init[0] = np.sin(beta * k_node * h) + np.zeros(shp(0))
    p.init[4] = A * np.cos(beta * k_cell * h) * math.sin(-wt * dt / 2) + np.zeros(shp(4))
    o = emo.Oracle(p)
    pts = np.asarray([[0, 1, 1, N], [0, 0, 0, 5], [0, 2, 2, N // 2]], np.int32)       # incl. the PMC wall k = N
    shape = np.sin(beta * pts[:, 3] * h)
    worst = 0.0
    for n in range(1, steps + 1):
        o.step(1)
        worst = max(worst, float(np.max(np.abs(o.probe(pts) - shape * math.cos(wt * n * dt)))))
    assert worst < 1e-11, worst
    f = o.fields()
    for c in (1, 2, 3, 5):
        assert np.all(f[c] == 0.0)
    # resonance: quarter-wave f = c0/(4L) up to the O(h^2) numerical dispersion
    f_cont = C0 / (4 * N * h)
    assert abs(wt / (2 * math.pi) / f_cont - 1) < 1e-3


def _energy_series(p, steps):
    """[energy^0 .. energy^steps] from E^n, H^{n-1/2}, H^{n+1/2}; the half dual
    lengths at the two ends of every axis are exactly the weights of PMC-wall edges"""
    o = emo.Oracle(p)
    geo = D.Geometry(p.dx, p.dy, p.dz)
    eps_e = [D.edge_mean(p.table[p.mat_id, 0], p.dx, p.dy, p.dz, a) for a in range(3)]
    nu_f = [D.face_mean(1.0 / p.table[p.mat_id, 1], p.dx, p.dy, p.dz, a) for a in range(3)]
    states = [o.fields()]
    for _ in range(steps + 1):
        o.step(1)
        states.append(o.fields())
    en = [D.energy(states[n][:3], states[n][3:], states[n + 1][3:], eps_e, nu_f, geo) for n in range(steps + 1)]
    return np.asarray(en), states


@pytest.mark.parametrize("bc", [(1, 1, 1, 1, 1, 1), (1, 0, 0, 1, 0, 1), (0, 1, 1, 0, 1, 0)])
def test_pmc_energy_conservation_mixed_walls(bc):
    p = W.random_problem(9, 7, 8, seed=41, lossless=True, n_ports=0, steps=400, bc=bc)
    en, states = _energy_series(p, 400)
    assert np.max(np.abs(en / en[0] - 1)) < 5e-13
    # the PMC walls carry field: tangential E on an all-PMC box is not zero
    if bc == (1, 1, 1, 1, 1, 1):
        assert np.max(np.abs(states[-1][0][0, :, :])) > 0 and np.max(np.abs(states[-1][2][:, :, 0])) > 0


def test_pmc_poynting_balance_with_wall_port():
    """energy^N - energy^0 + sum_c q_c V_c + dt sum_n sum_e Ebar_e J_e l_e A~_e = 0 (CD loss) with copper,
    a port on a PMC wall (dual area = the half face) and mixed walls"""
    steps = 300
    p = W.random_problem(8, 7, 6, seed=52, loss_mode=LOSS_CD, steps=steps, n_ports=2, init_scale=1.0e3,
                         bc=(0, 1, 1, 0, 0, 1))
    geo = D.Geometry(p.dx, p.dy, p.dz)
    en, states = _energy_series(p, steps)
    o = emo.Oracle(p); o.step(steps); _, q, Q = o.joule()
    work = 0.0
    for n in range(steps):
        for pt in range(p.n_ports):
            wv = p.wave[p.port_wave_offset[pt] + n] if n < p.port_wave_len[pt] else 0.0
            for e in range(p.port_edge_begin[pt], p.port_edge_end[pt]):
                c = int(p.edge_comp[e]); i, j, k = p.edge_ijk[e]
                eb = 0.5 * (states[n + 1][c][k, j, i] + states[n][c][k, j, i])
                work += p.dt * eb * p.port_amplitude[pt] * p.edge_weight[e] * wv * geo.len_e[c][k, j, i] * geo.area_dual[c][k, j, i]
    resid = en[steps] - en[0] + Q + work
    scale = max(abs(en[0]), abs(Q), abs(work))
    assert Q > 0 and abs(work) > 0
    assert abs(resid) < 2e-11 * scale, (resid, scale)


def test_pmc_rejects_unknown_bc_and_allows_wall_sources():
    p = W.random_problem(4, 4, 4, seed=61, n_ports=1, bc=(1, 0, 0, 0, 0, 0))
    emo.Oracle(p).step(2)                                     # the wall port is accepted
    p.bc = (2, 0, 0, 0, 0, 0)
    with pytest.raises(RuntimeError):
        emo.Oracle(p)
