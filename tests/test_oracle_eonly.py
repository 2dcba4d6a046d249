"""Pins of the E-only oracle (oracle/em_oracle_eonly.c: the paper's literal three-level recurrence, eq. (2)-(3),
PAPER.md L69-L76; NEXT-4 of SURVEY.md 8(f)).

None of these compares that oracle with itself:
  * the dense NumPy iteration of eq. (2)-(3) with matrices assembled from the incidence definition (tests/discrete.py),
    from RANDOM e^0 and e^{-1}, with sources and PMC walls;
  * the E/H leapfrog oracle (oracle/em_oracle.c, itself pinned by P0-P10), which eq. (2) reproduces exactly from
    (e^1, e^0) whatever H^{-1/2} was: heterogeneous non-uniform grids, CD and EXP, PMC walls;
  * the TE101 closed form: e^n = shape cos(w~ n dt) from e^0 = shape, e^{-1} = shape cos(w~ dt);
  * uniform conductor: e^n = r^n e^0 and the Joule geometric series (closed forms restated here).
"""
import math
import os

import numpy as np
import pytest

import workloads as W
from workloads.problem import LOSS_CD, LOSS_EXP, EPS0, MU0, C0
from oracle import emo
import discrete as D


@pytest.mark.parametrize("dims,seed,bc", [((4, 4, 4), 201, (0,) * 6), ((3, 5, 4), 202, (0,) * 6),
                                          ((4, 4, 4), 204, (1, 0, 0, 1, 1, 0)), ((3, 4, 5), 205, (1,) * 6)])
def test_dense_eq2_eq3_from_random_two_level_state(dims, seed, bc):
    nx, ny, nz = dims
    steps = 200
    p = W.random_problem(nx, ny, nz, seed=seed, loss_mode=LOSS_CD, steps=steps, n_ports=2, blocky=False, bc=bc)
    ops = D.Operators(nx, ny, nz, p.dx, p.dy, p.dz)
    eps_e = ops.flat([D.edge_mean(p.table[p.mat_id, 0], p.dx, p.dy, p.dz, a) for a in range(3)])
    sig_e = ops.flat([D.edge_mean(p.table[p.mat_id, 2], p.dx, p.dy, p.dz, a) for a in range(3)])
    nu_f = ops.flat([D.face_mean(1.0 / p.table[p.mat_id, 1], p.dx, p.dy, p.dz, a) for a in range(3)])
    free = ~ops.flat([D.fixed_mask(nx, ny, nz, a, bc=p.bc) for a in range(3)]).astype(bool)
    S = (ops.Ch.toarray() @ np.diag(nu_f) @ ops.Ce.toarray())[np.ix_(free, free)]
    dt = p.dt
    De, Ds = np.diag(eps_e[free]), np.diag(sig_e[free])
    M = De + 0.5 * dt * Ds; N = 2 * De - dt * dt * S; K = De - 0.5 * dt * Ds
    Minv = np.diag(1.0 / np.diag(M))

    def J_half(n):
        J = np.zeros(ops.eoff[-1])
        if n < 0:
            return J
        for pt in range(p.n_ports):
            w = p.wave[p.port_wave_offset[pt] + n] if n < p.port_wave_len[pt] else 0.0
            for e in range(p.port_edge_begin[pt], p.port_edge_end[pt]):
                c = int(p.edge_comp[e]); i, j, k = (int(v) for v in p.edge_ijk[e])
                J[ops.eidx(c, i, j, k)] += p.port_amplitude[pt] * p.edge_weight[e] * w
        return J

    rng = np.random.default_rng(seed + 1)
    e0 = [p.init[c] for c in range(3)]                       # random e^0 (all edges; fixed ones are forced to 0)
    em1 = [a + 0.05 * rng.standard_normal(a.shape) for a in e0]
    o = emo.OracleEOnly(p, e_prev=em1)
    e_cur = ops.flat(e0)[free]; e_prev = ops.flat(em1)[free]
    for n in range(steps):
        dJ = (J_half(n) - J_half(n - 1))[free] / dt
        e_next = Minv @ (N @ e_cur - K @ e_prev - dt * dt * dJ)
        e_prev, e_cur = e_cur, e_next
    o.step(steps)
    got = ops.flat(o.fields(0)); gotm = ops.flat(o.fields(1))
    assert np.all(got[~free] == 0.0)
    assert np.linalg.norm(got[free] - e_cur) <= 2e-12 * np.linalg.norm(e_cur)
    assert np.linalg.norm(gotm[free] - e_prev) <= 2e-12 * np.linalg.norm(e_prev)
    assert o.step_index == steps


@pytest.mark.parametrize("mode", [LOSS_CD, LOSS_EXP])
@pytest.mark.parametrize("dims,seed,bc", [((9, 7, 8), 301, (0,) * 6), ((6, 11, 5), 302, (1, 1, 1, 1, 0, 1)),
                                          ((1, 5, 7), 303, (0,) * 6), ((7, 6, 2), 304, (0, 1, 1, 0, 1, 1))])
def test_equals_the_leapfrog_oracle(dims, seed, bc, mode):
    """eq. (2) from (e^1, e^0) == the E/H leapfrog from (E^0, H^{-1/2}) for every later step; q likewise"""
    steps = 150
    p = W.random_problem(*dims, seed=seed, loss_mode=mode, steps=steps, n_ports=3, bc=bc)
    lf = emo.Oracle(p)
    E0 = lf.fields()[:3]
    lf.step(1)
    E1 = lf.fields()[:3]
    _, q1, _ = lf.joule()
    eo = emo.OracleEOnly(p, load_init=False)
    for c in range(3):
        eo.set_field(0, c, E1[c]); eo.set_field(1, c, E0[c])
    eo.set_step_index(1)
    for n in (1, 10, steps - 1):
        lf.step(n + 1 - lf.step_index); eo.step(n + 1 - eo.step_index)
        A, B = lf.fields()[:3], eo.fields(0)
        num = sum(float(np.sum((a - b) ** 2)) for a, b in zip(A, B)); den = sum(float(np.sum(a * a)) for a in A)
        assert num <= (1e-11) ** 2 * den, (n, (num / den) ** 0.5)
    pw_l, q_l, Q_l = lf.joule()
    pw_e, q_e, Q_e = eo.joule()
    assert np.max(np.abs((q_l - q1) - q_e)) <= 1e-10 * np.max(np.abs(q_l))
    assert np.max(np.abs(pw_l - pw_e)) <= 1e-10 * np.max(np.abs(pw_l))


def test_te101_closed_form_three_level():
    p = W.config1_cavity()
    n, h, dt = 16, 1.0e-3, p.dt
    s = math.sin(math.pi / (2 * n))
    w_num = (2.0 / dt) * math.asin(C0 * dt * math.sqrt(2 * s * s / (h * h)))
    e0 = [p.init.get(c, np.zeros(p.field_shape(c))) for c in range(3)]
    em1 = [a * math.cos(w_num * dt) for a in e0]             # the mode one step earlier (cos is even)
    o = emo.OracleEOnly(p, e_prev=em1)
    probe = [tuple(p.probes[0])]
    shape = math.sin(math.pi * 8 / n) * math.sin(math.pi * 8 / n)
    tr = [o.probe(probe)[0]]
    for _ in range(p.steps):
        o.step(1)
        tr.append(o.probe(probe)[0])
    tr = np.asarray(tr)
    want = shape * np.cos(w_num * np.arange(p.steps + 1) * dt)
    assert np.max(np.abs(tr - want)) < 1e-11                 # rounding grows like 1/sin(w dt) ~ 7 x the leapfrog's
    mid = np.abs(tr[1:-1]) > 0.2
    ratio = (tr[2:] + tr[:-2])[mid] / (2 * tr[1:-1][mid])
    assert abs(np.median(ratio) - math.cos(w_num * dt)) < 1e-12
    F = o.fields(0)
    assert np.all(F[0] == 0.0) and np.all(F[2] == 0.0)
    assert o.joule()[2] == 0.0


@pytest.mark.parametrize("mode", [LOSS_CD, LOSS_EXP])
def test_conductor_decay_and_joule_series(mode):
    nx, ny, nz, steps = 8, 7, 6, 300
    p = W.random_problem(nx, ny, nz, seed=41, loss_mode=mode, n_ports=0, steps=steps, ids=(1,))
    eps, sig = 11.9 * EPS0, 4.0e2
    p.table[1] = (eps, MU0, sig)
    p.dt = W.cfl_dt(p.dx, p.dy, p.dz, p.mat_id, p.table, 0.9)
    rng = np.random.default_rng(5)
    phi = np.zeros((nz + 1, ny + 1, nx + 1)); phi[1:-1, 1:-1, 1:-1] = rng.standard_normal((nz - 1, ny - 1, nx - 1))
    Ex = -(phi[:, :, 1:] - phi[:, :, :-1]) / p.dx[None, None, :]
    Ey = -(phi[:, 1:, :] - phi[:, :-1, :]) / p.dy[None, :, None]
    Ez = -(phi[1:, :, :] - phi[:-1, :, :]) / p.dz[:, None, None]
    x = sig * p.dt / (2 * eps)
    r = (1 - x) / (1 + x) if mode == LOSS_CD else math.exp(-2 * x)
    p.init = {0: Ex, 1: Ey, 2: Ez}
    o = emo.OracleEOnly(p, e_prev=[Ex / r, Ey / r, Ez / r])  # curl-free: S e = 0, so e^n = r^n e^0 solves eq. (2)
    o.step(steps)
    F = o.fields(0)
    rn = r ** steps
    for c, E0 in enumerate((Ex, Ey, Ez)):
        assert np.max(np.abs(F[c] - rn * E0)) < 1e-10 * np.max(np.abs(E0)) * rn

    def s_of(Ex, Ey, Ez):
        return 0.25 * (Ex[:-1, :-1, :] ** 2 + Ex[:-1, 1:, :] ** 2 + Ex[1:, :-1, :] ** 2 + Ex[1:, 1:, :] ** 2
                       + Ey[:-1, :, :-1] ** 2 + Ey[:-1, :, 1:] ** 2 + Ey[1:, :, :-1] ** 2 + Ey[1:, :, 1:] ** 2
                       + Ez[:, :-1, :-1] ** 2 + Ez[:, :-1, 1:] ** 2 + Ez[:, 1:, :-1] ** 2 + Ez[:, 1:, 1:] ** 2)
    s0 = s_of(Ex, Ey, Ez)
    pw, q, Q = o.joule()
    q_want = p.dt * sig * ((1 + r) / 2) ** 2 * (1 - r ** (2 * steps)) / (1 - r * r) * s0
    assert np.max(np.abs(q - q_want)) < 1e-11 * np.max(q_want)
    assert np.max(np.abs(pw - sig * r ** (2 * steps) * s0)) < 1e-9 * np.max(sig * r ** (2 * steps) * s0)
    geo = D.Geometry(p.dx, p.dy, p.dz)
    assert abs(Q - np.sum(q_want * geo.vol)) < 1e-11 * Q


def test_eonly_oracle_rejects_bad_arguments():
    p = W.random_problem(4, 4, 4, seed=71, n_ports=0)
    o = emo.OracleEOnly(p)
    with pytest.raises(RuntimeError):
        o.set_step_index(-1)
    with pytest.raises(RuntimeError):
        o.step(-1)
    bad = W.impulse_problem(); bad.edge_ijk = np.asarray([[2, 0, 1]], np.int32)      # a PEC-fixed edge
    with pytest.raises(RuntimeError):
        emo.OracleEOnly(bad)
    o.step(2); o.reset()
    assert o.step_index == 0 and not any(f.any() for f in o.fields(0))
