"""Pins of the oracle's thermal stage (NEXT-1 of SURVEY.md 8(f); eq. (4)-(6), L84-L96): forward-Euler heat
equation on the temperature rise theta = T - T0 per cell, driven by the Joule heat of the step, with the conductivity
feedback sigma(T) = sigma0 / (1 + alpha theta) refreshed every step.

Expected values are closed forms / invariants / an independently assembled operator, never the oracle itself:
 * adiabatic heating of a uniform lossy medium by a uniform decaying field: scalar recurrence + exact energy balance
   eps E^2/2 + rho c_p theta = const (CD loss);
 * pure diffusion of a cosine mode on a uniform grid: exact decay factor of the discrete Neumann Laplacian;
 * heat conservation and "heat gained == Joule energy lost by the field" on heterogeneous non-uniform grids;
 * M_kk assembled literally as V0a^T D_k V0 with dense matrices.
"""
import math

import numpy as np
import pytest

import workloads as W
from workloads.problem import LOSS_CD, LOSS_EXP, EPS0, MU0, C0, BC_PEC, BC_PMC, Problem
from oracle import emo


def _uniform_problem(nx, ny, nz, h, table, thermal, dt, bc=(0,) * 6, steps=0):
    d = lambda n, v: np.full(n, v)
    mat = np.zeros((nz, ny, nx), np.uint8)
    p = Problem("thermal_uniform", nx, ny, nz, d(nx, h[0]), d(ny, h[1]), d(nz, h[2]), mat,
                np.asarray(table, np.float64).reshape(1, 3), np.zeros(1, np.int32), dt, LOSS_CD, 64, steps)
    p.bc = tuple(bc)
    p.thermal = np.asarray(thermal, np.float64).reshape(1, 3)
    return p


@pytest.mark.parametrize("mode", [LOSS_CD, LOSS_EXP])
def test_adiabatic_uniform_heating_scalar_recurrence(mode):
    """Uniform Ex in a box whose y and z walls are PMC: curl E = 0, H stays 0, every cell is the same scalar
    problem.  Per step (paper order: D_sigma(T^n) in the E update L78, P^{n+1} into eq. (5), then eq. (6)):
        E' = ca(sigma_n) E,   dq = dt sigma_n ((E' + E)/2)^2,   theta += dq/(rho c_p),   sigma = sigma0/(1 + alpha theta)"""
    h = 1.0e-3
    dt = 0.9 * h / (C0 * math.sqrt(3.0))
    eps, sig0 = EPS0, 0.02 * EPS0 / dt * 5
    rho_cp, alpha, E0, steps = 1.0e3, 2.0, 1.0e7, 400
    p = _uniform_problem(3, 4, 3, (h, h, h), (eps, MU0, sig0), (rho_cp, 0.7, alpha), dt,
                         bc=(BC_PEC, BC_PEC, BC_PMC, BC_PMC, BC_PMC, BC_PMC))
    p.loss_mode = mode
    p.init = {0: np.full(p.field_shape(0), E0)}
    o = emo.Oracle(p)
    E, th, sg, q = E0, 0.0, sig0, 0.0
    for n in range(steps):
        if mode == LOSS_CD:
            x = sg * dt / (2 * eps); ca = (1 - x) / (1 + x)
        else:
            ca = math.exp(-sg * dt / eps)
        En = ca * E
        dq = dt * sg * (0.5 * (En + E)) ** 2
        q += dq; th += dq / rho_cp; sg = sig0 / (1 + alpha * th); E = En
    o.step(steps)
    f = o.fields()
    assert np.max(np.abs(f[0] / E - 1)) < 1e-12
    for c in range(1, 6):
        assert np.all(f[c] == 0.0)
    theta = o.temperature_rise()
    assert alpha * th > 0.3                                   # the feedback is strong, not a perturbation
    assert np.max(np.abs(theta / th - 1)) < 1e-12
    _, qm, _ = o.joule()
    assert np.max(np.abs(qm / q - 1)) < 1e-12
    if mode == LOSS_CD:                                       # exact discrete energy balance of eq. (2)-(3) + (5)
        assert abs((0.5 * eps * E * E + rho_cp * th) / (0.5 * eps * E0 * E0) - 1) < 1e-12
    # power density uses the CURRENT sigma(T)
    pw, _, _ = o.joule()
    assert np.max(np.abs(pw / (sg * E * E) - 1)) < 1e-12


def test_pure_diffusion_cosine_mode_closed_form():
    """sigma = 0, no field: theta^n = lambda^n theta^0 for theta^0 = prod_a cos(pi m_a (i_a + 1/2)/n_a), the DCT-II
    eigenvector of the cell-centred Neumann Laplacian: lambda = 1 - dt kappa sum_a (2 - 2 cos(pi m_a/n_a))/h_a^2"""
    nx, ny, nz = 8, 6, 5
    h = (1.0e-6, 1.5e-6, 0.8e-6)
    kth, rho_cp = 100.0, 2.0e6
    kappa = kth / rho_cp
    dt = 0.04 * min(h) ** 2 / kappa
    p = _uniform_problem(nx, ny, nz, h, (EPS0, MU0, 0.0), (rho_cp, kth, 0.0), dt)
    o = emo.Oracle(p)
    m = (3, 1, 2)
    ci = np.cos(math.pi * m[0] * (np.arange(nx) + 0.5) / nx)[None, None, :]
    cj = np.cos(math.pi * m[1] * (np.arange(ny) + 0.5) / ny)[None, :, None]
    ck = np.cos(math.pi * m[2] * (np.arange(nz) + 0.5) / nz)[:, None, None]
    th0 = 0.3 * ci * cj * ck
    o.set_temperature_rise(th0)
    lam = 1 - dt * kappa * sum((2 - 2 * math.cos(math.pi * m[a] / n)) / h[a] ** 2 for a, n in enumerate((nx, ny, nz)))
    assert 0.5 < lam < 0.95
    steps = 50
    o.step(steps)
    got = o.temperature_rise()
    assert np.max(np.abs(got - lam ** steps * th0)) < 1e-13 * np.max(np.abs(th0))


def _hetero_problem(seed, thermal_scale_k=1.0, alpha=True, **kw):
    p = W.random_problem(9, 7, 6, seed=seed, **kw)
    th = W.thermal_table()
    th[:, 1] *= thermal_scale_k
    if not alpha:
        th[:, 2] = 0.0
    p.thermal = th
    return p


def test_heat_gained_equals_joule_energy_and_diffusion_conserves_heat():
    """sum_c rho c_p theta_c V_c == Q = sum_c q_c V_c at every checkpoint (every joule deposited heats its own cell,
    conduction only moves heat between cells: flux antisymmetry, adiabatic walls), with sigma(T) feedback on,
    copper present, conduction exaggerated (k x 2e5) so that it matters at EM time steps, and one k = 0 material."""
    p = _hetero_problem(71, thermal_scale_k=2.0e5, steps=200, n_ports=2, init_scale=1.0e3)
    p.thermal[2, 1] = 0.0                                      # SiO2 cells do not conduct at all
    # explicit stability of eq. (5): dt * max(kappa) * sum 2/h^2 < 1 on this grid (exaggerated k)
    hmin = min(p.dx.min(), p.dy.min(), p.dz.min())
    assert p.dt * (p.thermal[:, 1] / p.thermal[:, 0]).max() * 6 / hmin ** 2 < 0.9
    o = emo.Oracle(p)
    vol = p.dz[:, None, None] * p.dy[None, :, None] * p.dx[None, None, :]
    rho_cp = p.thermal[p.mat_id, 0]
    prev = None
    for _ in range(4):
        o.step(50)
        th = o.temperature_rise()
        _, q, Q = o.joule()
        heat = float(np.sum(rho_cp * th * vol))
        assert Q > 0 and abs(heat / Q - 1) < 1e-11, (heat, Q)
        assert th.min() > -1e-12 * th.max()
        # conduction did move heat: theta differs from the adiabatic q / (rho c_p)
        assert np.linalg.norm(th - q / rho_cp) > 1e-3 * np.linalg.norm(th)
        prev = th


def test_sigma_feedback_changes_the_field_and_is_refreshed_every_step():
    """with alpha != 0 the run differs from the alpha = 0 run, and equals a run in which the test refreshes the
    temperature itself after every step through emo_set_temperature_rise (same numbers, different code path)"""
    kw = dict(steps=40, n_ports=2, init_scale=4.0e6)
    p = _hetero_problem(72, **kw)
    p.thermal[:, 2] *= 1.0e4                                   # exaggerated TCR: alpha theta ~ O(0.1) within 40 steps
    o = emo.Oracle(p); o.step(40)
    p0 = _hetero_problem(72, alpha=False, **kw)
    o0 = emo.Oracle(p0); o0.step(40)
    th = o.temperature_rise()
    assert (p.thermal[p.mat_id, 2] * th).max() > 0.02
    e, e0 = np.concatenate([a.ravel() for a in o.fields()[:3]]), np.concatenate([a.ravel() for a in o0.fields()[:3]])
    assert np.linalg.norm(e - e0) > 1e-4 * np.linalg.norm(e0)
    # manual refresh: run the alpha = 0 oracle one step at a time, but push sigma(T) in through a table whose
    # sigma0 is unchanged and a temperature field set by hand -> needs alpha != 0 in its table, adiabatic k
    p1 = _hetero_problem(72, **kw); p1.thermal[:, 2] *= 1.0e4
    o1 = emo.Oracle(p1)
    for _ in range(40):
        o1.step(1)
        o1.set_temperature_rise(o1.temperature_rise())          # idempotent refresh of sigma(T) and ca, cb
    e1 = np.concatenate([a.ravel() for a in o1.fields()[:3]])
    assert np.linalg.norm(e1 - e) <= 1e-14 * np.linalg.norm(e)


def test_mkk_is_v0a_t_dk_v0_dense():
    """One pure-diffusion step against M_kk = V0a^T D_k V0 assembled with dense matrices: V0 = negative
    gradient (cell difference / centre distance) on interior faces, D_k = series conductivity of the two half cells,
    V0a^T = divergence (face area / cell volume); heterogeneous materials, non-uniform spacings."""
    p = _hetero_problem(73, thermal_scale_k=2.0e5, steps=1, n_ports=0, lossless=True)
    p.init = None
    nx, ny, nz = p.nx, p.ny, p.nz
    d = [p.dx, p.dy, p.dz]
    k_c = p.thermal[p.mat_id, 1]; rho_cp = p.thermal[p.mat_id, 0]
    ncell = nx * ny * nz
    cid = lambda i, j, k: (k * ny + j) * nx + i
    rows = []                                                   # one row per interior face: (c, c', k_f, A_f, l_f)
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                for a, (di, dj, dk) in enumerate(((1, 0, 0), (0, 1, 0), (0, 0, 1))):
                    i2, j2, k2 = i + di, j + dj, k + dk
                    if i2 >= nx or j2 >= ny or k2 >= nz:
                        continue
                    idx, idx2 = (i, j, k)[a], (i2, j2, k2)[a]
                    la, lb = d[a][idx], d[a][idx2]
                    ka, kb = k_c[k, j, i], k_c[k2, j2, i2]
                    lf = 0.5 * (la + lb)
                    kf = lf / (0.5 * la / ka + 0.5 * lb / kb) if ka > 0 and kb > 0 else 0.0
                    area = np.prod([d[b][(i, j, k)[b]] for b in range(3) if b != a])
                    rows.append((cid(i, j, k), cid(i2, j2, k2), kf, area, lf))
    nf = len(rows)
    V0 = np.zeros((nf, ncell)); Dk = np.zeros((nf, nf)); DivT = np.zeros((ncell, nf))
    vol = (p.dz[:, None, None] * p.dy[None, :, None] * p.dx[None, None, :]).ravel()
    for f, (c1, c2, kf, area, lf) in enumerate(rows):
        V0[f, c1] = 1.0 / lf; V0[f, c2] = -1.0 / lf             # negative gradient along +axis
        Dk[f, f] = kf
        DivT[c1, f] = area / vol[c1]; DivT[c2, f] = -area / vol[c2]
    Mkk = DivT @ Dk @ V0
    assert np.max(np.abs(Mkk @ np.ones(ncell))) < 1e-6 * np.max(np.abs(Mkk))      # constants are in the null space
    rng = np.random.default_rng(5)
    th0 = rng.uniform(0.0, 1.0, size=(nz, ny, nx))
    o = emo.Oracle(p)
    o.set_temperature_rise(th0)
    o.step(1)
    want = th0.ravel() - p.dt / rho_cp.ravel() * (Mkk @ th0.ravel())
    got = o.temperature_rise().ravel()
    assert np.linalg.norm(want - th0.ravel()) > 1e-3 * np.linalg.norm(th0)          # the step is not a no-op
    assert np.linalg.norm(got - want) < 1e-13 * np.linalg.norm(want)


def test_thermal_argument_errors_and_reset():
    p = _hetero_problem(74, steps=5, n_ports=1)
    o = emo.Oracle(p)
    o.step(5)
    assert o.temperature_rise().max() > 0
    o.reset()
    assert np.all(o.temperature_rise() == 0.0)
    bad = p.thermal.copy(); bad[0, 0] = 0.0
    with pytest.raises(RuntimeError):
        o.set_thermal(bad)
    with pytest.raises(RuntimeError):
        o.set_temperature_rise(np.full((p.nz, p.ny, p.nx), -1.0e9))   # 1 + alpha theta <= 0 in copper
    p2 = W.random_problem(4, 4, 4, seed=75, n_ports=0)
    with pytest.raises(RuntimeError):
        emo.Oracle(p2).temperature_rise()                          # coupling not switched on
