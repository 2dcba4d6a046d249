"""GPU-vs-oracle parity of the two-way EM-thermal coupling (NEXT-1; eq. (4)-(6)) through the C ABI:
fields, Joule maps AND the temperature rise, element by element, same seeded inputs, tolerances of north_star."""
import numpy as np
import pytest

import workloads as W
from workloads.problem import LOSS_CD, LOSS_EXP
import paper_2603_07038_b200 as P
from oracle import emo
from parity import compare_state, rel_l2, TOL

pytestmark = pytest.mark.gpu


def _coupled(dims, seed, k_scale=2.0e5, tcr_scale=1.0e4, **kw):
    """random heterogeneous non-uniform grid with the thermal table; conduction and the temperature coefficient
    exaggerated so that both matter within a few dozen EM steps (see tests/test_oracle_thermal.py)"""
    p = W.random_problem(*dims, seed=seed, **kw)
    th = W.thermal_table()
    th[:, 1] *= k_scale; th[:, 2] *= tcr_scale
    p.thermal = th
    return p


STRATEGIES = [pytest.param(P.EM_KERNEL_AUTO, id="coupled-sweep"), pytest.param(P.EM_KERNEL_SPLIT, id="split")]


def _run(p, steps, precision, checkpoints=(), kernel=P.EM_KERNEL_AUTO, **em_kw):
    g = P.EM(p, precision=precision, kernel=kernel, **em_kw)
    o = emo.Oracle(p)
    tol = TOL[precision]
    done = 0
    for cp in list(checkpoints) + [steps]:
        g.em_step(cp - done); o.step(cp - done); done = cp
        res = compare_state(g, o, tol)
        tg, to = g.em_get_temperature_rise(), o.temperature_rise()
        res["theta"] = rel_l2([tg], [to])
        assert np.max(np.abs(to)) > 0
        assert res["theta"] <= tol, res
    g.close(); o.close()
    return res, to


CASES = [((37, 29, 23), LOSS_CD), ((9, 7, 6), LOSS_CD), ((130, 3, 2), LOSS_CD), ((1, 5, 7), LOSS_CD),
         ((37, 29, 23), LOSS_EXP), ((9, 7, 6), LOSS_EXP)]     # EXP on the non-degenerate grids, as in test_gpu_parity.py


@pytest.mark.parametrize("kernel", STRATEGIES)
@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("dims,mode", CASES)
def test_coupled_random_grids(dims, mode, precision, kernel):
    p = _coupled(dims, 8000 + sum(dims), loss_mode=mode, steps=60, n_ports=3, init_scale=4.0e6)
    res, theta = _run(p, 60, precision, checkpoints=(1, 10), kernel=kernel)
    # the feedback is not a perturbation below the tolerance: alpha * theta reaches the per-cent range
    assert (p.thermal[p.mat_id, 2] * theta).max() > 1e-3


@pytest.mark.parametrize("kernel", STRATEGIES)
def test_coupled_with_pmc_walls_and_wall_port(kernel):
    p = _coupled((21, 18, 12), 8101, steps=40, n_ports=4, init_scale=4.0e6, bc=(1, 1, 0, 1, 1, 1))
    _run(p, 40, 64, checkpoints=(1,), kernel=kernel)


@pytest.mark.parametrize("zsplit", [1, 3, 8])
def test_coupled_sweep_z_chunks(zsplit):
    p = _coupled((21, 18, 33), 8104, steps=30, n_ports=40, init_scale=4.0e6)
    _run(p, 30, 64, checkpoints=(1, 7), z_chunks=zsplit)


def test_pure_diffusion_and_set_get_temperature():
    p = _coupled((12, 9, 8), 8102, steps=30, n_ports=0, lossless=True)
    p.init = None
    rng = np.random.default_rng(9)
    th0 = rng.uniform(0.0, 1.0, size=(p.nz, p.ny, p.nx))
    for precision, kernel in ((64, P.EM_KERNEL_AUTO), (32, P.EM_KERNEL_AUTO), (64, P.EM_KERNEL_SPLIT)):
        g = P.EM(p, precision=precision, kernel=kernel); o = emo.Oracle(p)
        g.em_set_temperature_rise(th0); o.set_temperature_rise(th0)
        assert rel_l2([g.em_get_temperature_rise()], [th0]) <= (0 if precision == 64 else 1e-7)
        g.em_step(30); o.step(30)
        to = o.temperature_rise()
        assert np.linalg.norm(to - th0) > 1e-3 * np.linalg.norm(th0)
        assert rel_l2([g.em_get_temperature_rise()], [to]) <= TOL[precision]
        g.em_reset()
        assert not np.any(g.em_get_temperature_rise())
        g.close(); o.close()


def test_coupled_config4_scaled():
    """the package layout with the handbook-order thermal table as it stands (no exaggeration): tiny temperature
    rises, the coupled path must still match to tolerance"""
    p = W.make_config(4, scale=16, zscale=4, steps=80)
    p.thermal = W.thermal_table()
    for precision in (64, 32):
        _run(p, 80, precision)
    _run(p, 80, 32, kernel=P.EM_KERNEL_SPLIT)


def test_thermal_needs_flag_and_a_coupled_strategy():
    p = W.random_problem(6, 5, 4, seed=8103, n_ports=0)
    g = P.EM(p)
    with pytest.raises(P.EMError):
        g.em_set_thermal(W.thermal_table())                   # created with em_grid.thermal = 0
    with pytest.raises(P.EMError):
        g.em_get_temperature_rise()
    g.close()
    p.thermal = W.thermal_table()
    with pytest.raises(P.EMError):
        P.EM(p, formulation=P.EM_FORM_EONLY)                  # the E-only recurrence has no coupled variant
    bad = W.thermal_table(); bad[3, 2] = float("nan")
    p.thermal = bad
    with pytest.raises(P.EMError):
        P.EM(p)                                               # alpha must be finite


# ---- the NODAL thermal stage: theta on the mesh nodes, the paper's placement (em_grid.thermal = EM_THERMAL_NODE; N1-N4) ----
def _nodal(p):
    p.thermal_placement = "node"
    return p


NODAL_CASES = [(d, m, pr) for d, m in (((37, 29, 23), LOSS_CD), ((9, 7, 6), LOSS_EXP), ((130, 3, 2), LOSS_CD), ((1, 5, 7), LOSS_CD),
                                        ((2, 2, 2), LOSS_CD), ((33, 65, 4), LOSS_CD)) for pr in (64, 32)]


@pytest.mark.parametrize("dims,mode,precision", NODAL_CASES)
def test_nodal_coupled_random_grids(dims, mode, precision):
    p = _nodal(_coupled(dims, 8600 + sum(dims), loss_mode=mode, steps=60, n_ports=3 if min(dims) > 1 else 0, init_scale=4.0e6))
    res, theta = _run(p, 60, precision, checkpoints=(1, 10))
    assert theta.shape == (dims[2] + 1, dims[1] + 1, dims[0] + 1)
    if min(dims) > 2:
        assert np.abs(p.thermal[:, 2]).max() * np.abs(theta).max() > 1e-3        # the feedback is not below the tolerance


def test_nodal_with_pmc_walls_diffusion_and_api():
    p = _nodal(_coupled((21, 18, 12), 8601, steps=40, n_ports=4, init_scale=4.0e6, bc=(1, 1, 0, 1, 1, 1)))
    _run(p, 40, 64, checkpoints=(1,))
    # pure diffusion from a random nodal temperature, set / get / reset
    p = _nodal(_coupled((12, 9, 8), 8602, steps=30, n_ports=0, lossless=True))
    p.init = None
    th0 = np.random.default_rng(9).uniform(0.0, 1.0, size=(p.nz + 1, p.ny + 1, p.nx + 1))
    for precision in (64, 32):
        g = P.EM(p, precision=precision); o = emo.Oracle(p)
        g.em_set_temperature_rise(th0); o.set_temperature_rise(th0)
        g.em_step(30); o.step(30)
        to = o.temperature_rise()
        assert np.linalg.norm(to - th0) > 1e-3 * np.linalg.norm(th0)
        assert rel_l2([g.em_get_temperature_rise()], [to]) <= TOL[precision]
        g.em_reset()
        assert not np.any(g.em_get_temperature_rise())
        g.close(); o.close()
    with pytest.raises(P.EMError) as e:
        P.EM(p, kernel=P.EM_KERNEL_TMA)                       # the nodal stage runs on the split kernels
    assert e.value.code == 5


def test_nodal_paper_mesh_unknown_count_and_package_slice():
    """config 6 scaled: (nx+1)(ny+1)(nz+1) temperature unknowns (full size: 377 x 409 x 46 = 7 092 878)"""
    p = _nodal(W.make_config(6, scale=8, steps=40))
    p.thermal = W.thermal_table()
    res, theta = _run(p, 40, 32)
    assert theta.size == (p.nx + 1) * (p.ny + 1) * (p.nz + 1) and 377 * 409 * 46 == 7092878
