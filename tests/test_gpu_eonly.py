"""GPU parity of the E-only three-level recurrence (em_grid.formulation = EM_FORM_EONLY; NEXT-4 of SURVEY.md 8(f);
PAPER.md L69 eq. (2), L73-L76 eq. (3)) against its own oracle (oracle/em_oracle_eonly.c), through the C ABI.

Tolerances.  The recurrence feeds every rounding error delta of a stored e into the difference e^n - e^{n-1}, i.e. into
the "velocity"; a mode of temporal frequency w then carries it with the gain 1/sin(w dt) instead of 1 (DESIGN.md,
E-only section).  Two independent roundings of the same recurrence (GPU, oracle) therefore differ by about
sqrt(n) eps / (w dt) after n steps, not sqrt(n) eps:
  fp64: 1e-11 for the runs here (measured 1e-15 .. 5e-13);
  fp32: 2e-5 holds only for short runs (<= 100 steps); the long run records what it reaches and asserts only that the
        error stays below 1e-2 -- it does NOT meet north_star's 2e-5 at 1000 steps, which is why LEAPFROG is the default.
"""
import math

import numpy as np
import pytest

import workloads as W
from workloads.problem import LOSS_CD, LOSS_EXP, C0
import paper_2603_07038_b200 as P
from oracle import emo
from parity import max_norm_err, rel_l2

pytestmark = pytest.mark.gpu

TOL_EO = {64: 1e-11, 32: 2e-5}


def compare_eonly(g, o, tol):
    Fg, Fo = g.fields(), o.fields(0) + o.fields(1)
    res = dict(e=rel_l2(Fg[:3], Fo[:3]), em=rel_l2(Fg[3:], Fo[3:]), emax=max_norm_err(Fg[:3], Fo[:3]))
    pg, qg, Qg = g.joule_maps()
    po, qo, Qo = o.joule()
    res.update(q=rel_l2([qg], [qo]), p=rel_l2([pg], [po]), Q=abs(Qg - Qo) / abs(Qo) if Qo != 0 else abs(Qg),
               qmax=max_norm_err([qg], [qo]))
    assert res["e"] <= tol and res["em"] <= tol and res["emax"] <= tol, res
    assert res["q"] <= tol and res["Q"] <= tol and res["p"] <= 2 * tol and res["qmax"] <= tol, res
    return res


def run_pair(p, steps, precision, checkpoints=(), tol=None, seed=1, **em_kw):
    rng = np.random.default_rng(seed)
    e_prev = None
    if p.init:
        e_prev = [p.init[c] + 0.05 * rng.standard_normal(p.init[c].shape) for c in range(3)]
    g = P.EM(p, precision=precision, formulation=P.EM_FORM_EONLY, e_prev=e_prev, **em_kw)
    o = emo.OracleEOnly(p, e_prev=e_prev)
    tol = tol or TOL_EO[precision]
    done = 0
    res = None
    for cp in list(checkpoints) + [steps]:
        g.em_step(cp - done); o.step(cp - done); done = cp
        res = compare_eonly(g, o, tol)
    assert g.step_index == steps
    g.close(); o.close()
    return res


SMALL = [(37, 29, 23), (1, 5, 7), (130, 3, 2), (5, 1, 9), (6, 7, 1), (1, 1, 1), (33, 65, 4), (64, 17, 40)]


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("dims", SMALL)
def test_random_grids_cd(dims, precision):
    p = W.random_problem(*dims, seed=1000 + sum(dims), loss_mode=LOSS_CD, steps=40, n_ports=3)
    run_pair(p, 40, precision, checkpoints=(1, 10))


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("dims", [(37, 29, 23), (9, 4, 70)])
def test_random_grids_exp(dims, precision):
    p = W.random_problem(*dims, seed=2000 + sum(dims), loss_mode=LOSS_EXP, steps=40, n_ports=3)
    run_pair(p, 40, precision, checkpoints=(1,))


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("bc", [(1, 1, 1, 1, 1, 1), (1, 0, 0, 1, 0, 1), (0, 1, 1, 0, 1, 0)])
@pytest.mark.parametrize("dims", [(37, 29, 23), (33, 65, 4)])
def test_random_grids_pmc_walls(dims, bc, precision):
    p = W.random_problem(*dims, seed=5000 + sum(dims) + sum(bc), loss_mode=LOSS_CD, steps=40, n_ports=3, bc=bc)
    run_pair(p, 40, precision, checkpoints=(1, 10))


@pytest.mark.parametrize("zsplit", [1, 2, 3, 5, 8])
def test_z_chunks_and_many_ports(zsplit):
    p = W.random_problem(21, 18, 33, seed=78, loss_mode=LOSS_CD, steps=30, n_ports=60, bc=(0, 0, 1, 0, 1, 1))
    run_pair(p, 30, 64, checkpoints=(1, 7), z_chunks=zsplit)


def test_percell_ids_pec_material_and_uniform_mu():
    p = W.random_problem(21, 19, 17, seed=3001, blocky=False, steps=30, n_ports=2)
    run_pair(p, 30, 64)
    p = W.random_problem(21, 19, 17, seed=3002, pec_material=True, steps=30, n_ports=0)
    run_pair(p, 30, 64)
    p = W.random_problem(21, 19, 17, seed=3004, steps=30, n_ports=2, ids=(0, 1, 2, 3))      # uniform mu fast path
    run_pair(p, 30, 64)


def test_config1_te101_three_level():
    """e^0 = the mode, e^{-1} = the mode one step earlier: e^n = shape cos(w~ n dt) (closed form, 1000 steps)"""
    p = W.config1_cavity()
    n, h, dt = 16, 1.0e-3, p.dt
    s = math.sin(math.pi / (2 * n))
    w_num = (2.0 / dt) * math.asin(C0 * dt * math.sqrt(2 * s * s / (h * h)))
    e0 = [p.init.get(c, np.zeros(p.field_shape(c))) for c in range(3)]
    em1 = [a * math.cos(w_num * dt) for a in e0]
    p.init = {c: e0[c] for c in range(3)}
    g = P.EM(p, precision=64, formulation=P.EM_FORM_EONLY, e_prev=em1)
    o = emo.OracleEOnly(p, e_prev=em1)
    tr = [g.em_probe(p.probes)[0]]
    for _ in range(10):
        g.em_step(100); o.step(100)
        tr.append(g.em_probe(p.probes)[0])
    want = np.cos(w_num * dt * 100 * np.arange(11))
    assert np.max(np.abs(np.asarray(tr) - want)) < 2e-11
    res = compare_eonly(g, o, 1e-11)
    assert res["Q"] == 0.0
    g.close()


def test_equals_the_leapfrog_kernel():
    """the E-only context started from (E^1, E^0) of a leapfrog context reproduces its E for every later step"""
    p = W.random_problem(37, 29, 23, seed=6001, steps=60, n_ports=3, bc=(0, 1, 0, 0, 1, 0))
    lf = P.EM(p, precision=64)
    E0 = [lf.em_get_field(c) for c in range(3)]
    lf.em_step(1)
    E1 = [lf.em_get_field(c) for c in range(3)]
    eo = P.EM(p, precision=64, formulation=P.EM_FORM_EONLY, load_init=False)
    for c in range(3):
        eo.em_set_field(c, E0[c])
    eo.em_step(1)                       # only to move the step index to 1 (the waveform sample the next step uses) ...
    for c in range(3):
        eo.em_set_field(c, E1[c]); eo.em_set_field(6 + c, E0[c])     # ... then impose the state (e^1, e^0)
    lf.em_step(59); eo.em_step(59)
    A = [lf.em_get_field(c) for c in range(3)]; B = [eo.em_get_field(c) for c in range(3)]
    assert rel_l2(B, A) <= 1e-11
    with pytest.raises(P.EMError):
        eo.em_get_field(3)              # an E-only context has no H
    with pytest.raises(P.EMError):
        lf.em_get_field(6)
    lf.close(); eo.close()


def test_config4_scaled_1000_steps_fp64_and_what_fp32_reaches():
    """config 4 at 1/8 of the x, y cell counts for its stated 1000 steps: fp64 within 1e-11; fp32 recorded (it leaves
    the 2e-5 bound: rounding errors of e enter e^n - e^{n-1} and are amplified by ~1/(w dt))"""
    p = W.make_config(4, scale=8, steps=1000)
    res64 = run_pair(p, 1000, 64)
    g = P.EM(p, precision=32, formulation=P.EM_FORM_EONLY)
    o = emo.OracleEOnly(p)
    errs = []
    for _ in range(10):
        g.em_step(100); o.step(100)
        errs.append(rel_l2(g.fields()[:3], o.fields(0)))
    print("E-only config 4 (1/8): fp64", res64, " fp32 rel-L2(e) every 100 steps:", ["%.1e" % e for e in errs])
    assert errs[0] <= 2e-5              # 100 steps: still inside the fp32 bound
    assert errs[-1] <= 1e-2             # 1000 steps: degraded, bounded (measured ~2e-4)
    g.close(); o.close()
