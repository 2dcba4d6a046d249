"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these compares the oracle with itself: expected values are closed forms, invariants,
hand-derived numbers (tests/golden/) or independently assembled operators (tests/discrete.py).
"""
import math
import os

import numpy as np
import pytest

import workloads as W
from workloads.problem import LOSS_CD, LOSS_EXP, EPS0, MU0, C0
from oracle import emo
import discrete as D

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _read_kv(path):
    kv, rows = {}, []
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        parts = line.split()
        if len(parts) == 2:
            kv[parts[0]] = parts[1]
        else:
            rows.append(parts)
    return kv, rows


# ------------------------------------------------------------------------------------------ P0
def test_p0_dof_counts():
    """EM DOF = #edges of the 376x408x45 mesh; thermal = #nodes; mech = 3 #nodes."""
    kv, _ = _read_kv(os.path.join(GOLD, "paper_dof.txt"))
    nx, ny, nz = int(kv["nx"]), int(kv["ny"]), int(kv["nz"])
    sh = D.shapes(nx, ny, nz)
    assert sum(int(np.prod(s)) for s in sh[:3]) == int(kv["em_dof"])
    assert (nx + 1) * (ny + 1) * (nz + 1) == int(kv["thermal_dof"])
    assert 3 * (nx + 1) * (ny + 1) * (nz + 1) == int(kv["mechanical_dof"])
    # and the oracle's arrays have exactly these logical extents
    p = W.random_problem(5, 4, 3, seed=0, n_ports=0)
    o = emo.Oracle(p)
    assert [o.get_field(c).shape for c in range(6)] == D.shapes(5, 4, 3)


# ----------------------------------------------------------------------------------------- P10
def test_p10_impulse_worked_example():
    kv, rows = _read_kv(os.path.join(GOLD, "impulse_4x4x4.txt"))
    p = W.impulse_problem()
    assert abs(p.dt - float(kv["dt"])) < 1e-24
    a, S2, h = p.dt / EPS0, float(kv["S2"]), float(kv["h"])
    assert abs(a - float(kv["a"])) < 1e-14
    assert abs((C0 * p.dt / h) ** 2 - S2) < 1e-15
    o = emo.Oracle(p)
    names = {"Ex": 0, "Ey": 1, "Ez": 2, "Hx": 3, "Hy": 4, "Hz": 5}
    for step in (1, 2, 3):
        o.step(1)
        F = o.fields()
        listed = {c: set() for c in range(6)}
        for r in rows:
            if int(r[0]) != step:
                continue
            c = names[r[1]]; i, j, k = int(r[2]), int(r[3]), int(r[4])
            want = eval(r[5], {"a": a, "S2": S2, "h": h})
            got = F[c][k, j, i]
            assert abs(got - want) <= 1e-12 * max(abs(want), 1e-30) + 1e-18, (step, r, got, want)
            listed[c].add((k, j, i))
        if step in (1, 2):   # the file lists every non-zero entry for steps 1 and 2
            for c in range(6):
                nz_idx = set(map(tuple, np.argwhere(F[c] != 0.0)))
                assert nz_idx == listed[c], (step, c, nz_idx ^ listed[c])
        if step == 3:
            assert np.count_nonzero(F[3]) == 12 and np.count_nonzero(F[4]) == 12
            assert np.count_nonzero(F[5]) == 0
            assert abs(F[0].sum()) < 1e-15 and abs(F[1].sum()) < 1e-15


# ------------------------------------------------------------------------------------------ P1
def test_p1_te101_closed_form():
    kv, _ = _read_kv(os.path.join(GOLD, "te101.txt"))
    p = W.config1_cavity()
    n, h, dt = 16, 1.0e-3, p.dt
    assert abs(dt - float(kv["dt"])) < 1e-20
    s = math.sin(math.pi / (2 * n))
    w_num = (2.0 / dt) * math.asin(C0 * dt * math.sqrt(2 * s * s / (h * h)))
    f_cont = 0.5 * C0 * math.sqrt(2.0 / (n * h) ** 2)
    assert abs(f_cont / 1e9 - float(kv["f101_continuous_GHz"])) < 1e-5
    assert abs(w_num / (2 * math.pi) / 1e9 - float(kv["f101_numerical_GHz"])) < 1e-8
    assert abs(math.cos(w_num * dt) - float(kv["cos_w_dt"])) < 1e-14
    o = emo.Oracle(p)
    probe = [tuple(p.probes[0])]
    shape = math.sin(math.pi * 8 / n) * math.sin(math.pi * 8 / n)
    tr = [o.probe(probe)[0]]
    for _ in range(p.steps):
        o.step(1)
        tr.append(o.probe(probe)[0])
    tr = np.asarray(tr)
    nn = np.arange(p.steps + 1)
    want = shape * np.cos(w_num * nn * dt)
    assert np.max(np.abs(tr - want)) < 2e-12
    # resonance from the trace itself: three-term ratio (E^{n+1} + E^{n-1}) / 2E^n = cos(w dt)
    mid = np.abs(tr[1:-1]) > 0.2
    ratio = (tr[2:] + tr[:-2])[mid] / (2 * tr[1:-1][mid])
    f_meas = np.arccos(np.median(ratio)) / dt / (2 * math.pi)
    assert abs(f_meas / (w_num / 2 / math.pi) - 1) < 1e-10
    assert abs(f_meas / f_cont - 1) < 1e-3          # O(h^2) dispersion, -0.074 %
    F = o.fields()
    for c in (0, 2, 4):                              # spurious components stay exactly zero
        assert np.all(F[c] == 0.0)
    _, q, Q = o.joule()
    assert Q == 0.0 and np.all(q == 0.0)


def _energy_series(p, steps, eps_eff=None):
    """[energy^0 .. energy^steps] using E^n, H^{n-1/2}, H^{n+1/2} (trial step = the next step)."""
    o = emo.Oracle(p)
    geo = D.Geometry(p.dx, p.dy, p.dz)
    eps_c = p.table[p.mat_id, 0]; nu_c = 1.0 / p.table[p.mat_id, 1]
    eps_e = eps_eff if eps_eff is not None else [D.edge_mean(eps_c, p.dx, p.dy, p.dz, a) for a in range(3)]
    nu_f = [D.face_mean(nu_c, p.dx, p.dy, p.dz, a) for a in range(3)]
    states = [o.fields()]
    for _ in range(steps + 1):
        o.step(1)
        states.append(o.fields())
    en = []
    for n in range(steps + 1):
        E = states[n][:3]; Hm = states[n][3:]; Hp = states[n + 1][3:]
        en.append(D.energy(E, Hm, Hp, eps_e, nu_f, geo))
    return np.asarray(en), states, o


# ------------------------------------------------------------------------------------------ P2
def test_p2_energy_conservation_cavity():
    kv, _ = _read_kv(os.path.join(GOLD, "te101.txt"))
    p = W.config1_cavity(steps=300)
    en, _, _ = _energy_series(p, 300)
    assert np.max(np.abs(en / en[0] - 1)) < 1e-12
    assert abs(en[0] / float(kv["energy_J"]) - 1) < 1e-6


@pytest.mark.parametrize("seed", [11, 12])
def test_p2_energy_conservation_heterogeneous_nonuniform(seed):
    p = W.random_problem(9, 7, 8, seed=seed, lossless=True, n_ports=0, steps=400)
    en, _, _ = _energy_series(p, 400)
    assert np.max(np.abs(en / en[0] - 1)) < 5e-13


# ------------------------------------------------------------------------------------------ P3
@pytest.mark.parametrize("mode", [LOSS_CD, LOSS_EXP])
def test_p3_poynting_balance(mode):
    """energy^N - energy^0 + sum_c q_c V_c + dt sum_n sum_e Ebar_e J_e l_e A~_e = 0 with copper and
    sources present; EXP uses the effective permittivity eps' = (s dt/2) coth(s dt / 2 eps)."""
    steps = 300
    p = W.random_problem(8, 7, 6, seed=21 + mode, loss_mode=mode, steps=steps, n_ports=2, init_scale=1.0e3)
    geo = D.Geometry(p.dx, p.dy, p.dz)
    eps_c = p.table[p.mat_id, 0]; sig_c = p.table[p.mat_id, 2]
    eps_e = [D.edge_mean(eps_c, p.dx, p.dy, p.dz, a) for a in range(3)]
    sig_e = [D.edge_mean(sig_c, p.dx, p.dy, p.dz, a) for a in range(3)]
    if mode == LOSS_EXP:
        eff = []
        for a in range(3):
            x = sig_e[a] * p.dt / (2 * eps_e[a])
            with np.errstate(divide="ignore", invalid="ignore", over="ignore"):
                e2 = np.where(x > 1e-9, (sig_e[a] * p.dt / 2) / np.tanh(x), eps_e[a] * (1 + x * x / 3))
            eff.append(e2)
        eps_e = eff
    en, states, o = _energy_series(p, steps, eps_eff=eps_e)
    _, q, Q = o.joule()
    # q from the oracle covers steps+1 steps (the trial step); recompute work up to `steps` only
    o2 = emo.Oracle(p); o2.step(steps); _, q, Q = o2.joule()
    src_work = 0.0
    for n in range(steps):
        for pt in range(p.n_ports):
            wv = p.wave[p.port_wave_offset[pt] + n] if n < p.port_wave_len[pt] else 0.0
            for e in range(p.port_edge_begin[pt], p.port_edge_end[pt]):
                c = int(p.edge_comp[e]); i, j, k = p.edge_ijk[e]
                J = p.port_amplitude[pt] * p.edge_weight[e] * wv
                eb = 0.5 * (states[n + 1][c][k, j, i] + states[n][c][k, j, i])
                src_work += p.dt * eb * J * geo.len_e[c][k, j, i] * geo.area_dual[c][k, j, i]
    resid = en[steps] - en[0] + Q + src_work
    scale = max(abs(en[0]), abs(Q), abs(src_work))
    assert abs(Q - float(np.sum(q * geo.vol))) <= 1e-12 * abs(Q)
    assert Q > 0
    assert abs(resid) < 2e-11 * scale, (resid, scale, en[0], Q, src_work)


# ------------------------------------------------------------------------------------------ P4
def test_p4_divergence_invariants():
    steps = 60
    p = W.random_problem(7, 6, 8, seed=31, lossless=True, n_ports=2, steps=steps)
    nx, ny, nz = p.nx, p.ny, p.nz
    geo = D.Geometry(p.dx, p.dy, p.dz)
    eps_e = [D.edge_mean(p.table[p.mat_id, 0], p.dx, p.dy, p.dz, a) for a in range(3)]
    nu_f = [D.face_mean(1.0 / p.table[p.mat_id, 1], p.dx, p.dy, p.dz, a) for a in range(3)]

    def div_b(H):
        fx = H[0] / nu_f[0] * geo.area_f[0]; fy = H[1] / nu_f[1] * geo.area_f[1]; fz = H[2] / nu_f[2] * geo.area_f[2]
        return (fx[:, :, 1:] - fx[:, :, :-1]) + (fy[:, 1:, :] - fy[:, :-1, :]) + (fz[1:, :, :] - fz[:-1, :, :])

    def div_d(E):   # at interior nodes (1..n-1)^3
        fx = eps_e[0] * E[0] * geo.area_dual[0]; fy = eps_e[1] * E[1] * geo.area_dual[1]; fz = eps_e[2] * E[2] * geo.area_dual[2]
        return ((fx[1:-1, 1:-1, 1:] - fx[1:-1, 1:-1, :-1]) + (fy[1:-1, 1:, 1:-1] - fy[1:-1, :-1, 1:-1])
                + (fz[1:, 1:-1, 1:-1] - fz[:-1, 1:-1, 1:-1]))

    o = emo.Oracle(p)
    F0 = o.fields()
    o.step(steps)
    F1 = o.fields()
    b0, b1 = div_b(F0[3:]), div_b(F1[3:])
    scale_b = max(np.max(np.abs(F[3] / nu_f[0] * geo.area_f[0])) for F in (F0, F1))
    assert np.max(np.abs(b1 - b0)) < 1e-12 * scale_b
    d0, d1 = div_d(F0[:3]), div_d(F1[:3])
    touched = np.zeros((nz + 1, ny + 1, nx + 1), bool)       # nodes touched by a source edge
    for e in range(len(p.edge_comp)):
        c = int(p.edge_comp[e]); i, j, k = (int(v) for v in p.edge_ijk[e])
        touched[k, j, i] = True
        touched[k + (c == 2), j + (c == 1), i + (c == 0)] = True
    free = ~touched[1:-1, 1:-1, 1:-1]
    scale_d = max(np.max(np.abs(eps_e[0] * F[0] * geo.area_dual[0])) for F in (F0, F1))
    assert free.sum() > 50
    assert np.max(np.abs((d1 - d0)[free])) < 1e-11 * scale_d
    assert np.max(np.abs((d1 - d0)[~free])) > 1e-6 * scale_d   # and the sources do inject charge


# --------------------------------------------------------------------------------------- P5, P6
@pytest.mark.parametrize("mode", [LOSS_CD, LOSS_EXP])
def test_p5_p6_conductor_decay_and_joule_series(mode):
    nx, ny, nz, steps = 8, 7, 6, 400
    p = W.random_problem(nx, ny, nz, seed=41, loss_mode=mode, n_ports=0, steps=steps, ids=(1,))
    eps, sig = 11.9 * EPS0, 4.0e2
    p.table[1] = (eps, MU0, sig)
    p.dt = W.cfl_dt(p.dx, p.dy, p.dz, p.mat_id, p.table, 0.9)
    rng = np.random.default_rng(5)
    phi = np.zeros((nz + 1, ny + 1, nx + 1)); phi[1:-1, 1:-1, 1:-1] = rng.standard_normal((nz - 1, ny - 1, nx - 1))
    Ex = -(phi[:, :, 1:] - phi[:, :, :-1]) / p.dx[None, None, :]
    Ey = -(phi[:, 1:, :] - phi[:, :-1, :]) / p.dy[None, :, None]
    Ez = -(phi[1:, :, :] - phi[:-1, :, :]) / p.dz[:, None, None]
    sh = D.shapes(nx, ny, nz)
    p.init = {0: Ex, 1: Ey, 2: Ez, 3: np.zeros(sh[3]), 4: np.zeros(sh[4]), 5: np.zeros(sh[5])}
    x = sig * p.dt / (2 * eps)
    r = (1 - x) / (1 + x) if mode == LOSS_CD else math.exp(-2 * x)
    o = emo.Oracle(p)
    o.step(steps)
    F = o.fields()
    rn = r ** steps
    for c, E0 in enumerate((Ex, Ey, Ez)):
        assert np.max(np.abs(F[c] - rn * E0)) < 1e-12 * np.max(np.abs(E0)) * max(rn, 1e-3) + 1e-13 * rn
    for c in (3, 4, 5):                    # curl-free E never excites H
        assert np.max(np.abs(F[c])) < 1e-12 * np.max(np.abs(Ex)) / 377.0
    if mode == LOSS_CD:                    # CD agrees with exp(-sigma t/eps) to O(x^3) per step
        assert abs(math.log(r) + 2 * x) < 2 * x ** 3
    # P6: Joule geometric series and instantaneous power
    def s_of(Ex, Ey, Ez):
        return 0.25 * (Ex[:-1, :-1, :] ** 2 + Ex[:-1, 1:, :] ** 2 + Ex[1:, :-1, :] ** 2 + Ex[1:, 1:, :] ** 2
                       + Ey[:-1, :, :-1] ** 2 + Ey[:-1, :, 1:] ** 2 + Ey[1:, :, :-1] ** 2 + Ey[1:, :, 1:] ** 2
                       + Ez[:, :-1, :-1] ** 2 + Ez[:, :-1, 1:] ** 2 + Ez[:, 1:, :-1] ** 2 + Ez[:, 1:, 1:] ** 2)
    s0 = s_of(Ex, Ey, Ez)
    pw, q, Q = o.joule()
    q_want = p.dt * sig * ((1 + r) / 2) ** 2 * (1 - r ** (2 * steps)) / (1 - r * r) * s0
    assert np.max(np.abs(q - q_want)) < 1e-12 * np.max(q_want)
    assert np.max(np.abs(pw - sig * r ** (2 * steps) * s0)) < 1e-11 * np.max(sig * r ** (2 * steps) * s0)
    geo = D.Geometry(p.dx, p.dy, p.dz)
    assert abs(Q - np.sum(q_want * geo.vol)) < 1e-12 * Q
    if mode == LOSS_CD:                    # all the initial electric energy ends up as heat
        e0 = 0.5 * eps * sum(np.sum(E ** 2 * geo.len_e[c] * geo.area_dual[c]) for c, E in enumerate((Ex, Ey, Ez)))
        assert abs(Q - e0 * (1 - r ** (2 * steps))) < 1e-11 * e0


# ------------------------------------------------------------------------------------------ P8
@pytest.mark.parametrize("mode", [LOSS_CD, LOSS_EXP])
def test_p8_cyclic_axis_permutation(mode):
    """(x', y', z') = (y, z, x): E'x = Ey, E'y = Ez, E'z = Ex (same for H); arrays transpose(2,0,1)."""
    steps = 25
    p = W.random_problem(6, 5, 7, seed=51, loss_mode=mode, n_ports=3, steps=steps)
    T = lambda a: np.ascontiguousarray(np.transpose(a, (2, 0, 1)))
    import copy
    r = copy.copy(p)
    r.nx, r.ny, r.nz = p.ny, p.nz, p.nx
    r.dx, r.dy, r.dz = p.dy.copy(), p.dz.copy(), p.dx.copy()
    r.mat_id = T(p.mat_id)
    cmap = {0: 2, 1: 0, 2: 1}               # old component -> new component
    r.init = {}
    for c in range(3):
        r.init[cmap[c]] = T(p.init[c]); r.init[3 + cmap[c]] = T(p.init[3 + c])
    r.edge_comp = np.asarray([cmap[int(c)] for c in p.edge_comp], np.int32)
    r.edge_ijk = np.asarray([(j, k, i) for (i, j, k) in p.edge_ijk], np.int32).reshape(-1, 3)
    a, b = emo.Oracle(p), emo.Oracle(r)
    a.step(steps); b.step(steps)
    Fa, Fb = a.fields(), b.fields()
    for c in range(3):
        for off in (0, 3):
            x, y = T(Fa[off + c]), Fb[off + cmap[c]]
            assert np.max(np.abs(x - y)) <= 1e-12 * np.max(np.abs(x))
    qa, qb = a.joule()[1], b.joule()[1]
    assert np.max(np.abs(T(qa) - qb)) <= 1e-12 * np.max(qa)


# ------------------------------------------------------------------------------------------ P9
def test_p9_cfl_rule_vs_power_iteration():
    """dt_rule(f=1) <= 2/sqrt(lambda_max(D_eps^-1 S)) on a graded heterogeneous lossless grid."""
    import scipy.sparse as sp
    import scipy.sparse.linalg as spl
    rng = np.random.default_rng(61)
    nx, ny, nz = 12, 10, 9
    g = lambda n: 0.5e-6 * 1.2 ** np.abs(np.arange(n) - n // 2)
    dx, dy, dz = g(nx), g(ny), g(nz)
    p = W.random_problem(nx, ny, nz, seed=61, lossless=True, n_ports=0)
    p.dx, p.dy, p.dz = dx, dy, dz
    dt1 = emo.cfl_dt(nx, ny, nz, dx, dy, dz, p.mat_id, p.table)
    assert abs(dt1 - W.cfl_dt(dx, dy, dz, p.mat_id, p.table, 1.0)) < 1e-12 * dt1
    ops = D.Operators(nx, ny, nz, dx, dy, dz)
    eps_e = ops.flat([D.edge_mean(p.table[p.mat_id, 0], dx, dy, dz, a) for a in range(3)])
    nu_f = ops.flat([D.face_mean(1.0 / p.table[p.mat_id, 1], dx, dy, dz, a) for a in range(3)])
    free = ~ops.flat([D.fixed_mask(nx, ny, nz, a) for a in range(3)]).astype(bool)
    S = (ops.Ch @ sp.diags(nu_f) @ ops.Ce).tocsr()[free][:, free]
    A = sp.diags(1.0 / eps_e[free]) @ S
    lam = spl.eigs(A, k=1, which="LM", return_eigenvectors=False, tol=1e-8)[0].real
    dt_true = 2.0 / math.sqrt(lam)
    assert dt1 <= dt_true
    assert dt1 > 0.5 * dt_true


def test_p9b_cfl_rule_hand_computed_2x2x2():
    """absolute anchor of emo_cfl_dt on a non-uniform two-material grid: the hand-computed minimum of
    tests/golden/cfl_2x2x2.txt (the material decides which cell wins, so a wrong min/max, exponent or index order fails)"""
    kv, _ = _read_kv(os.path.join(GOLD, "cfl_2x2x2.txt"))
    dx, dy, dz = np.asarray([1e-3, 2e-3]), np.asarray([1e-3, 3e-3]), np.asarray([2e-3, 1e-3])
    table = np.asarray([[EPS0, MU0, 0.0], [4.0 * EPS0, MU0, 0.0]])
    mat = np.zeros((2, 2, 2), np.uint8); mat[1, 0, 0] = 1                 # [k][j][i]: cell (i, j, k) = (0, 0, 1)
    got = emo.cfl_dt(2, 2, 2, dx, dy, dz, mat, table)
    assert abs(got - float(kv["dt_max"])) <= 1e-13 * got
    assert abs(W.cfl_dt(dx, dy, dz, mat, table, 1.0) - float(kv["dt_max"])) <= 1e-13 * got
    mat[:] = 0
    got = emo.cfl_dt(2, 2, 2, dx, dy, dz, mat, table)
    assert abs(got - float(kv["dt_max_if_cell_001_were_vacuum"])) <= 1e-13 * got


# --------------------------------------------------------------------------- API / edge cases
def test_oracle_rejects_bad_arguments():
    p = W.random_problem(4, 4, 4, seed=71, n_ports=0)
    o = emo.Oracle(p)
    p2 = W.impulse_problem()
    p2.edge_ijk = np.asarray([[2, 0, 1]], np.int32)         # Ez on the -y wall: PEC-fixed
    with pytest.raises(RuntimeError):
        emo.Oracle(p2)
    bad = W.random_problem(4, 4, 4, seed=72, n_ports=0)
    bad.mat_id[0, 0, 0] = 200
    with pytest.raises(RuntimeError):
        emo.Oracle(bad)
    o.step(0)
    assert o.step_index == 0


def test_oracle_reset_restarts_the_run_exactly():
    """emo_reset zeroes the six fields, q and the step counter (waveform index): the rerun repeats the first run bit for bit"""
    p = W.random_problem(7, 6, 5, seed=72, n_ports=3, steps=25)
    p.init = None
    o = emo.Oracle(p)
    o.step(25)
    first = o.fields(); _, q1, Q1 = o.joule()
    assert any(f.any() for f in first) and Q1 > 0
    o.reset()
    assert o.step_index == 0 and not any(f.any() for f in o.fields())
    _, q0, Q0 = o.joule()
    assert Q0 == 0.0 and not q0.any()
    o.step(25)
    again = o.fields(); _, q2, Q2 = o.joule()
    assert all(np.array_equal(a, b) for a, b in zip(first, again)) and np.array_equal(q1, q2) and Q1 == Q2


def test_oracle_pec_material_edges_stay_zero():
    p = W.random_problem(7, 6, 5, seed=81, pec_material=True, n_ports=0, steps=10)
    pec = (p.flags[p.mat_id] & 1).astype(bool)
    assert pec.any()
    o = emo.Oracle(p); o.step(10)
    F = o.fields()
    for c in range(3):
        m = D.fixed_mask(p.nx, p.ny, p.nz, c, pec)
        assert np.all(F[c][m] == 0.0)
        assert np.any(F[c][~m] != 0.0)


def test_degenerate_dims_run():
    for dims in [(1, 5, 7), (6, 1, 4), (5, 4, 1), (1, 1, 1), (2, 2, 2)]:
        p = W.random_problem(*dims, seed=91, n_ports=1, steps=5)
        o = emo.Oracle(p); o.step(5)
        F = o.fields()
        assert all(np.all(np.isfinite(f)) for f in F)
