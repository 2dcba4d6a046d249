"""Pins of the oracle's NODAL thermal stage -- the paper's placement of T (7 092 878 thermal unknowns = the
nodes of its 376 x 408 x 45 mesh; eq. (4)-(6) L84-L96; M_kk = V0a^T D_k V0, L86), readings N1-N4 of DESIGN.md section 9.

Expected values are the paper's printed count, closed forms, invariants and an independently assembled operator:
 * the unknown count on the paper's mesh (tests/golden/paper_dof.txt);
 * one diffusion step against M_kk assembled literally, with dense matrices, as (V~)^-1 B^T diag(k_e A~_e / l_e) B
   (B = the signed node-to-edge incidence, i.e. V0 l), on heterogeneous non-uniform grids with a k = 0 material;
 * pure diffusion of a cosine mode on a uniform grid: exact decay factor of the nodal Neumann Laplacian (half dual cells
   at the walls, i.e. the DCT-I modes);
 * adiabatic heating of a uniform lossy medium by a uniform decaying field: the scalar recurrence, every node alike;
 * heat gained by the nodes == Joule energy the field lost == the per-cell Joule map's total, step by step."""
import math
import os

import numpy as np
import pytest

import workloads as W
from workloads.problem import LOSS_CD, LOSS_EXP, EPS0, MU0, C0, BC_PEC, BC_PMC, Problem
from oracle import emo

HERE = os.path.dirname(os.path.abspath(__file__))


def _nodal(p):
    p.thermal_placement = "node"
    return p


def _uniform_problem(nx, ny, nz, h, table, thermal, dt, bc=(0,) * 6):
    d = lambda n, v: np.full(n, v)
    p = Problem("thermal_uniform_nodal", nx, ny, nz, d(nx, h[0]), d(ny, h[1]), d(nz, h[2]), np.zeros((nz, ny, nx), np.uint8),
                np.asarray(table, np.float64).reshape(1, 3), np.zeros(1, np.int32), dt, LOSS_CD, 64, 0)
    p.bc = tuple(bc)
    p.thermal = np.asarray(thermal, np.float64).reshape(1, 3)
    return _nodal(p)


def test_unknown_count_of_the_papers_mesh():
    gold = dict(l.split() for l in open(os.path.join(HERE, "golden", "paper_dof.txt")) if l.strip() and not l.startswith("#"))
    nx, ny, nz = int(gold["nx"]), int(gold["ny"]), int(gold["nz"])
    assert (nx + 1) * (ny + 1) * (nz + 1) == int(gold["thermal_dof"]) == 7092878
    p = _nodal(W.random_problem(5, 4, 3, seed=1, n_ports=0))
    p.thermal = W.thermal_table()
    o = emo.Oracle(p)
    assert o.temperature_rise().shape == (4, 5, 6) and o.temperature_rise().size == 6 * 5 * 4
    o.close()


def _dense_operator(p):
    """(C, K): nodal heat capacities [J/K] and the conductance matrix [W/K] K = B^T diag(k_e A~_e / l_e) B, assembled edge
    by edge from the cells (nothing shared with the oracle: own loops, own indexing)."""
    nx, ny, nz = p.nx, p.ny, p.nz
    d = (np.asarray(p.dx), np.asarray(p.dy), np.asarray(p.dz))
    kc = p.thermal[p.mat_id, 1]; rc = p.thermal[p.mat_id, 0]
    nid = lambda i, j, k: (k * (ny + 1) + j) * (nx + 1) + i
    nn = (nx + 1) * (ny + 1) * (nz + 1)
    K = np.zeros((nn, nn)); Cn = np.zeros(nn)
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                vol = d[0][i] * d[1][j] * d[2][k]
                for dk in (0, 1):
                    for dj in (0, 1):
                        for di in (0, 1):
                            Cn[nid(i + di, j + dj, k + dk)] += rc[k, j, i] * vol / 8.0
                # the 12 edges of the cell: each gets a quarter of the cell's cross-section normal to it
                for axis in range(3):
                    o1, o2 = [a for a in range(3) if a != axis]
                    area = d[o1][(i, j, k)[o1]] * d[o2][(i, j, k)[o2]]
                    g = kc[k, j, i] * area / 4.0 / d[axis][(i, j, k)[axis]]
                    for s1 in (0, 1):
                        for s2 in (0, 1):
                            a = [i, j, k]; a[o1] += s1; a[o2] += s2
                            b = list(a); b[axis] += 1
                            na, nb = nid(*a), nid(*b)
                            K[na, na] += g; K[nb, nb] += g; K[na, nb] -= g; K[nb, na] -= g
    return Cn, K


@pytest.mark.parametrize("dims,seed", [((4, 3, 5), 3), ((2, 2, 2), 4), ((1, 4, 3), 5), ((6, 1, 1), 6)])
def test_one_diffusion_step_against_the_dense_v0at_dk_v0(dims, seed):
    p = _nodal(W.random_problem(*dims, seed=seed, n_ports=0, lossless=True))
    th = W.thermal_table(); th[:, 1] *= 3.0e4
    th[1, 1] = 0.0                                           # one material that does not conduct
    p.thermal = th; p.init = None
    o = emo.Oracle(p)
    rng = np.random.default_rng(seed)
    t0 = rng.uniform(-1.0, 1.0, size=o.theta_shape)
    o.set_temperature_rise(t0)
    o.step(1)
    Cn, K = _dense_operator(p)
    want = t0.ravel() - p.dt * (K @ t0.ravel()) / Cn
    got = o.temperature_rise().ravel()
    assert np.linalg.norm(want - t0.ravel()) > 1e-6 * np.linalg.norm(t0)          # the step moved something
    assert np.max(np.abs(got - want)) <= 1e-13 * np.max(np.abs(t0))
    assert abs(np.dot(Cn, got) - np.dot(Cn, t0.ravel())) <= 1e-13 * np.dot(Cn, np.abs(t0.ravel()))     # heat is conserved
    o.close()


def test_cosine_mode_decay_closed_form():
    nx, ny, nz, h = 6, 5, 4, (1.0e-6, 1.5e-6, 2.0e-6)
    rho_cp, kth = 1.6e6, 150.0
    dt = 0.9 * h[0] / (C0 * math.sqrt(3.0))
    p = _uniform_problem(nx, ny, nz, h, (EPS0, MU0, 0.0), (rho_cp, kth * 2.0e5, 0.0), dt)
    kk = kth * 2.0e5
    o = emo.Oracle(p)
    m = (2, 1, 3)
    i, j, k = np.meshgrid(np.arange(nx + 1), np.arange(ny + 1), np.arange(nz + 1), indexing="ij")
    mode = (np.cos(math.pi * m[0] * i / nx) * np.cos(math.pi * m[1] * j / ny) * np.cos(math.pi * m[2] * k / nz)).transpose(2, 1, 0)
    o.set_temperature_rise(mode)
    lam = 1.0 - dt * kk / rho_cp * sum(2.0 / h[a] ** 2 * (1.0 - math.cos(math.pi * m[a] / n)) for a, n in enumerate((nx, ny, nz)))
    assert 0.0 < lam < 0.999
    steps = 50
    o.step(steps)
    assert np.max(np.abs(o.temperature_rise() - lam ** steps * mode)) <= 1e-12
    o.close()


@pytest.mark.parametrize("mode", [LOSS_CD, LOSS_EXP])
def test_adiabatic_uniform_heating_scalar_recurrence(mode):
    """uniform Ex between PMC walls in y and z: every edge carries the same field, every node heats alike (wall nodes have
    half / quarter dual volumes AND half / quarter edge shares), so the nodal stage is the cell stage's scalar recurrence"""
    h = 1.0e-3
    dt = 0.9 * h / (C0 * math.sqrt(3.0))
    eps, sig0 = EPS0, 0.1 * EPS0 / dt
    rho_cp, alpha, E0, steps = 1.0e3, 2.0, 1.0e7, 300
    p = _uniform_problem(3, 4, 3, (h, h, h), (eps, MU0, sig0), (rho_cp, 0.7, alpha), dt, bc=(BC_PEC, BC_PEC, BC_PMC, BC_PMC, BC_PMC, BC_PMC))
    p.loss_mode = mode
    p.init = {0: np.full(p.field_shape(0), E0)}
    o = emo.Oracle(p)
    E, th, sg = E0, 0.0, sig0
    for n in range(steps):
        if mode == LOSS_CD:
            x = sg * dt / (2 * eps); ca = (1 - x) / (1 + x)
        else:
            ca = math.exp(-sg * dt / eps)
        En = ca * E
        th += dt * sg * (0.5 * (En + E)) ** 2 / rho_cp; sg = sig0 / (1 + alpha * th); E = En
    o.step(steps)
    theta = o.temperature_rise()
    assert alpha * th > 0.3                                   # the feedback matters
    assert np.max(np.abs(o.fields()[0] / E - 1)) < 1e-12
    # the x walls are PEC but Ex is normal to them: every node, wall nodes included, sees the same heating
    assert np.max(np.abs(theta / th - 1)) < 1e-12
    o.close()


@pytest.mark.parametrize("mode", [LOSS_CD, LOSS_EXP])
def test_heat_gained_by_the_nodes_is_the_joule_energy(mode):
    p = _nodal(W.random_problem(7, 5, 6, seed=21, loss_mode=mode, steps=30, n_ports=3, bc=(0, 1, 0, 0, 1, 0), init_scale=4.0e6))
    th = W.thermal_table(); th[:, 1] *= 2.0e5; th[:, 2] *= 1.0e4
    p.thermal = th
    o = emo.Oracle(p)
    Cn, _ = _dense_operator(p)
    vol = np.asarray(p.dz)[:, None, None] * np.asarray(p.dy)[None, :, None] * np.asarray(p.dx)[None, None, :]
    heat_prev = Q_prev = 0.0
    for n in range(30):
        o.step(1)
        heat = float(np.dot(Cn, o.temperature_rise().ravel()))
        _, q, Q = o.joule()
        assert abs(Q - float(np.sum(q * vol))) <= 1e-12 * Q
        assert abs((heat - heat_prev) - (Q - Q_prev)) <= 1e-10 * Q           # per step: conduction moves heat, only Joule adds it
        heat_prev, Q_prev = heat, Q
    assert Q > 0 and np.max(np.abs(p.thermal[p.mat_id, 2])) * np.max(o.temperature_rise()) > 1e-3
    o.close()
