"""GPU-vs-oracle parity (all through the C ABI).  Tolerances are BASELINE.json north_star's:
relative L2 <= 1e-12 (fp64) and <= 2e-5 (fp32) for E, H, the Joule map and the Joule total."""
import math
import os

import numpy as np
import pytest

import workloads as W
from workloads.problem import LOSS_CD, LOSS_EXP, C0
import paper_2603_07038_b200 as P
from oracle import emo
from parity import TOL, compare_state, rel_l2, subbox_problem

pytestmark = pytest.mark.gpu

KERNELS = [pytest.param(P.EM_KERNEL_SPLIT, id="split"), pytest.param(P.EM_KERNEL_TMA, id="tma")]


def run_pair(p, steps, precision, kernel, checkpoints=(), **em_kw):
    g = P.EM(p, precision=precision, kernel=kernel, **em_kw)
    o = emo.Oracle(p)
    tol = TOL[precision]
    done = 0
    res = None
    for cp in list(checkpoints) + [steps]:
        g.em_step(cp - done); o.step(cp - done); done = cp
        res = compare_state(g, o, tol)
    assert g.step_index == steps
    g.close(); o.close()
    return res


# ------------------------------------------------------------------------------ worked examples
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("precision", [64, 32])
def test_impulse_example(kernel, precision):
    p = W.impulse_problem()
    run_pair(p, 3, precision, kernel, checkpoints=(1, 2))


@pytest.mark.parametrize("kernel", KERNELS)
def test_config1_cavity_te101(kernel):
    """config 1: 16^3 PEC cavity, fp64, 1000 steps; also checks the GPU against the closed form."""
    p = W.config1_cavity()
    g = P.EM(p, precision=64, kernel=kernel)
    o = emo.Oracle(p)
    n, h, dt = 16, 1.0e-3, p.dt
    s = math.sin(math.pi / (2 * n))
    w_num = (2.0 / dt) * math.asin(C0 * dt * math.sqrt(2 * s * s / (h * h)))
    tr = [g.em_probe(p.probes)[0]]
    for _ in range(10):
        g.em_step(100); o.step(100)
        tr.append(g.em_probe(p.probes)[0])
    want = np.cos(w_num * dt * 100 * np.arange(11))
    assert np.max(np.abs(np.asarray(tr) - want)) < 2e-12
    res = compare_state(g, o, 1e-12)
    assert res["Q"] == 0.0
    g.close()


# ------------------------------------------------------------- randomised heterogeneous grids
SMALL = [(37, 29, 23), (1, 5, 7), (130, 3, 2), (5, 1, 9), (6, 7, 1), (1, 1, 1), (2, 2, 2), (33, 65, 4), (64, 17, 40)]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("dims", SMALL)
def test_random_grids_cd(dims, precision, kernel):
    p = W.random_problem(*dims, seed=1000 + sum(dims), loss_mode=LOSS_CD, steps=40, n_ports=3)
    run_pair(p, 40, precision, kernel, checkpoints=(1, 10))


@pytest.mark.parametrize("zsplit", [1, 2, 3, 5, 8])
@pytest.mark.parametrize("bc", [(0,) * 6, (0, 0, 1, 0, 1, 1)])
def test_tma_sweep_z_chunks(zsplit, bc):
    """The sweep splits every tile column into z chunks (work items; em_grid.z_chunks forces the count); many ports so
    that source edges sit on chunk boundary planes (their E' closes the Joule sum of the chunk below)."""
    p = W.random_problem(21, 18, 33, seed=78, loss_mode=LOSS_CD, steps=30, n_ports=60, bc=bc)
    run_pair(p, 30, 64, P.EM_KERNEL_TMA, checkpoints=(1, 7), z_chunks=zsplit)


def test_tma_sweep_is_deterministic_across_runs_and_chunkings():
    """The TMA sweep has no CTA barrier in its plane loop (mbarrier / named-barrier hand-offs between rows): a missing
    ordering would show up as run-to-run or chunking-dependent bits.  256 x 256 x 192 package slice, 228 work items
    and more, 40 steps, fp32: every run must give IDENTICAL bits."""
    p = W.make_config(4, scale=4, steps=40)
    ref = None
    for zsplit in (3, 3, 1, 8, 3):
        g = P.EM(p, precision=32, kernel=P.EM_KERNEL_TMA, z_chunks=zsplit)
        g.em_step(40)
        out = [g.em_get_field(c) for c in range(6)] + [g.joule_maps()[1]]
        g.close()
        if ref is None:
            ref = out
            assert all(np.isfinite(a).all() for a in out) and np.abs(out[0]).max() > 0
        else:
            for a, b in zip(out, ref):
                assert np.array_equal(a, b), zsplit


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("dims", [(37, 29, 23), (9, 4, 70)])
def test_random_grids_exp(dims, precision, kernel):
    p = W.random_problem(*dims, seed=2000 + sum(dims), loss_mode=LOSS_EXP, steps=40, n_ports=3)
    run_pair(p, 40, precision, kernel, checkpoints=(1,))


# --------------------------------------------------------------------- PMC walls
PMC_BC = [(1, 1, 1, 1, 1, 1), (1, 0, 0, 1, 0, 1), (0, 1, 1, 0, 1, 0), (1, 1, 1, 1, 0, 1)]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("bc", PMC_BC)
@pytest.mark.parametrize("dims", [(37, 29, 23), (130, 3, 2), (5, 9, 2), (33, 65, 4)])
def test_random_grids_pmc_walls(dims, bc, precision, kernel):
    """per-face PMC walls (tangential E of the wall updated with the half dual face), one port ON a PMC wall,
    random initial fields that are non-zero on the PMC walls"""
    p = W.random_problem(*dims, seed=5000 + sum(dims) + sum(bc), loss_mode=LOSS_CD, steps=40, n_ports=3, bc=bc)
    run_pair(p, 40, precision, kernel, checkpoints=(1, 10))


@pytest.mark.parametrize("kernel", KERNELS)
def test_pmc_exp_loss_and_z_chunks(kernel):
    p = W.random_problem(21, 18, 33, seed=5101, loss_mode=LOSS_EXP, steps=30, n_ports=20, bc=(0, 1, 1, 1, 1, 1))
    run_pair(p, 30, 64, kernel, checkpoints=(1, 7), z_chunks=3)


@pytest.mark.parametrize("kernel", KERNELS)
def test_config6_paper_mesh_scaled(kernel):
    """the paper-shaped run (PAPER.md L160 mesh, 20 fs, PEC ground + PMC walls) at 1/4 of the x, y cell counts"""
    p = W.make_config(6, scale=4, steps=300)
    assert p.bc == (1, 1, 1, 1, 0, 1) and p.dt == 20.0e-15
    run_pair(p, 300, 32, kernel, checkpoints=(10,))


def test_config6_paper_mesh_full_size():
    """376 x 408 x 45 cells = the paper's 21 088 285 EM unknowns, fp32, AUTO strategy, the whole field compared"""
    p = W.make_config(6, steps=120)
    ne = p.nx * (p.ny + 1) * (p.nz + 1) + (p.nx + 1) * p.ny * (p.nz + 1) + (p.nx + 1) * (p.ny + 1) * p.nz
    assert ne == 21088285
    run_pair(p, 120, 32, P.EM_KERNEL_AUTO, checkpoints=(3,))


@pytest.mark.parametrize("kernel", KERNELS)
def test_random_grid_percell_ids_and_pec_material(kernel):
    p = W.random_problem(21, 19, 17, seed=3001, blocky=False, steps=30, n_ports=2)
    run_pair(p, 30, 64, kernel)
    p = W.random_problem(21, 19, 17, seed=3002, pec_material=True, steps=30, n_ports=0)
    run_pair(p, 30, 64, kernel)


@pytest.mark.parametrize("kernel", KERNELS)
def test_overlapping_ports_add(kernel):
    p = W.random_problem(9, 8, 7, seed=3003, steps=12, n_ports=2)
    # make port 1 drive the same edges as port 0 (contributions add, C14)
    e0 = slice(int(p.port_edge_begin[0]), int(p.port_edge_end[0]))
    n0 = e0.stop - e0.start
    p.edge_comp = np.concatenate([p.edge_comp[e0], p.edge_comp[e0]])
    p.edge_ijk = np.concatenate([p.edge_ijk[e0], p.edge_ijk[e0]])
    p.edge_weight = np.concatenate([p.edge_weight[e0], -0.5 * p.edge_weight[e0]])
    p.port_edge_begin = np.asarray([0, n0], np.int64); p.port_edge_end = np.asarray([n0, 2 * n0], np.int64)
    run_pair(p, 12, 64, kernel)


# --------------------------------------------------------------------- the five configurations
@pytest.mark.parametrize("kernel", KERNELS)
def test_config2_slab_scaled_full_steps(kernel):
    """config 2 at 32x32x64 (oracle in seconds), all 5000 steps, fp64, EXP loss."""
    p = W.make_config(2, scale=4)
    res = run_pair(p, p.steps, 64, kernel, checkpoints=(1, 10))
    assert res["Q"] <= 1e-12


def test_config2_slab_full_size():
    """config 2 at its full 128x128x64 size, 250 steps (bounded for the oracle)."""
    p = W.make_config(2, steps=250)
    run_pair(p, 250, 64, P.EM_KERNEL_AUTO)


@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("kappa", [1.0, 100.0])
def test_config3_interposer_scaled(precision, kappa):
    p = W.make_config(3, scale=4, steps=400, kappa=kappa, precision=precision)
    run_pair(p, 400, precision, P.EM_KERNEL_AUTO, checkpoints=(10,))


@pytest.mark.parametrize("kernel", KERNELS)
def test_config4_package_scaled(kernel):
    p = W.make_config(4, scale=8, zscale=2, steps=300)
    g = P.EM(p, precision=32, kernel=kernel)
    o = emo.Oracle(p)
    for _ in range(3):                    # Joule map output every 100 steps, as in the config
        g.em_step(100); o.step(100)
        compare_state(g, o, TOL[32])
    g.close()


def test_config5_graded_scaled():
    p = W.make_config(5, scale=8, zscale=4, steps=300)
    assert p.dx.max() / p.dx.min() > 20
    run_pair(p, 300, 32, P.EM_KERNEL_AUTO, checkpoints=(10,))
    run_pair(p, 100, 64, P.EM_KERNEL_AUTO)


# ------------------------------------------------- full BASELINE sizes: sampled light-cone parity
def _fullsize_sampled(cfg, precision, n_steps=3, n_boxes=4, half=7, **kw):
    """At the full configuration size in the launch configuration bench.py times: random device
    initial state, n_steps on the GPU, then every output inside a few sample boxes is recomputed by
    the oracle on the box enlarged by the domain of dependence (n_steps + 2 cells)."""
    import torch
    p = W.make_config(cfg, **kw)
    g = P.EM(p, precision=precision, kernel=P.EM_KERNEL_AUTO)
    gen = torch.Generator(device="cuda"); gen.manual_seed(1234 + cfg)
    shapes = g.shapes
    init = []
    for c in range(6):
        t = torch.randn(shapes[c], generator=gen, device="cuda", dtype=g.dtype)
        if c >= 3:
            t /= 376.73
        g.em_set_field(c, t)
        init.append(g.em_get_field(c, device=True).clone())     # after PEC masking
        del t
    g.em_step(n_steps)
    out = [g.em_get_field(c, device=True) for c in range(6)]
    qmap = torch.empty((p.nz, p.ny, p.nx), dtype=g.dtype, device="cuda")
    g.em_joule(None, qmap, total=False)
    rng = np.random.default_rng(77 + cfg)
    m = n_steps + 2
    centres = []
    if p.n_ports:                                                 # boxes at port edges first
        for q in rng.choice(p.n_ports, size=min(2, p.n_ports), replace=False):
            centres.append(tuple(int(v) for v in p.edge_ijk[int(p.port_edge_begin[q])]))
    while len(centres) < n_boxes:
        centres.append((int(rng.integers(0, p.nx)), int(rng.integers(0, p.ny)), int(rng.integers(0, p.nz))))
    centres.append((0, 0, 0)); centres.append((p.nx - 1, p.ny - 1, p.nz - 1))
    worst = 0.0
    for (ci, cj, ck) in centres:
        core_lo = [max(0, ci - half), max(0, cj - half), max(0, ck - half)]
        core_hi = [min(p.nx, ci + half), min(p.ny, cj + half), min(p.nz, ck + half)]
        lo = [max(0, v - m) for v in core_lo]
        hi = [min(n, v + m) for v, n in zip(core_hi, (p.nx, p.ny, p.nz))]
        (i0, j0, k0), (i1, j1, k1) = lo, hi
        ext = [(0, 1, 1), (1, 0, 1), (1, 1, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1)]     # +1 per axis (x, y, z)
        sub = lambda arr, c: arr[k0:k1 + ext[c][2], j0:j1 + ext[c][1], i0:i1 + ext[c][0]].cpu().numpy()
        bp = subbox_problem(p, lo, hi, [sub(init[c], c) for c in range(6)])
        o = emo.Oracle(bp)
        o.step(n_steps)
        Fo = o.fields()
        _, qo, _ = o.joule()
        # compare only the core (unaffected by the artificial PEC walls of the box)
        a = [core_lo[d] - lo[d] for d in range(3)]; b = [core_hi[d] - lo[d] for d in range(3)]
        sl = lambda f: f[a[2]:b[2], a[1]:b[1], a[0]:b[0]]
        got = [sl(sub(out[c], c)) for c in range(6)]
        want = [sl(Fo[c]) for c in range(6)]
        eE = rel_l2(got[:3], want[:3]); eH = rel_l2(got[3:], want[3:])
        qg = qmap[k0:k1, j0:j1, i0:i1].cpu().numpy()
        eq = rel_l2([sl(qg)], [sl(qo)])
        worst = max(worst, eE, eH, eq)
        assert eE <= TOL[precision] and eH <= TOL[precision] and eq <= TOL[precision], ((ci, cj, ck), eE, eH, eq)
    g.close()
    return worst


def test_fullsize_sampled_config3_fp32():
    _fullsize_sampled(3, 32)


def test_fullsize_sampled_config3_fp64():
    _fullsize_sampled(3, 64)


def test_fullsize_sampled_config4_fp32():
    _fullsize_sampled(4, 32)


def test_fullsize_sampled_config5_fp32():
    _fullsize_sampled(5, 32)


# ------------------------------------------------------------------------------ C-ABI contract
def test_api_contract():
    p = W.random_problem(12, 11, 10, seed=4001, steps=10, n_ports=2)
    g = P.EM(p, precision=64)
    F0 = g.fields()
    g.em_step(0)
    assert g.step_index == 0 and all(np.array_equal(a, b) for a, b in zip(F0, g.fields()))
    # PEC-fixed tangential E is forced to 0 on set
    assert np.all(F0[0][:, 0, :] == 0) and np.all(F0[0][0, :, :] == 0) and np.all(F0[2][:, :, 0] == 0)
    # bad arguments
    with pytest.raises(P.EMError):
        g.em_probe([(0, p.nx, 0, 0)])
    with pytest.raises(P.EMError):
        g.em_step(-1)
    bad = W.impulse_problem(); bad.edge_ijk = np.asarray([[2, 0, 1]], np.int32)
    with pytest.raises(P.EMError):
        P.EM(bad)
    # capacities
    with pytest.raises(P.EMError) as e:
        P.EM(p, max_source_edges=1)
    assert e.value.code == 2
    # reset semantics of em_joule and em_reset
    g.em_step(5)
    _, q1, Q1 = g.joule_maps(reset=True)
    _, q2, Q2 = g.joule_maps()
    assert Q1 > 0 and Q2 == 0.0 and not q2.any()
    g.em_reset()
    assert g.step_index == 0 and not any(f.any() for f in g.fields())
    # two contexts coexist; repeated create/destroy
    for _ in range(3):
        a, b = P.EM(p, precision=64), P.EM(p, precision=32)
        a.em_step(2); b.em_step(2)
        assert rel_l2(b.fields()[:3], a.fields()[:3]) < 1e-5
        a.close(); b.close()
    g.close()


def test_probe_matches_fields():
    p = W.random_problem(10, 9, 8, seed=4002, steps=5, n_ports=1)
    g = P.EM(p, precision=64)
    g.em_step(5)
    F = g.fields()
    vals = g.em_probe(p.probes)
    for v, (c, i, j, k) in zip(vals, p.probes):
        assert v == F[c][k, j, i]
    g.close()


def test_configs_4_and_5_at_their_stated_1000_steps():
    """BASELINE.json: parity "after the stated step count".  The package configs at 1/4 (config 4) and 1/8 (config 5)
    of the x, y cell counts, full z, full 1000 steps, fp32, AUTO strategy: measured rel-L2 4e-7 (E), 2e-6 (H), 5e-7 (q)."""
    for cfg, kw in ((4, dict(scale=4)), (5, dict(scale=8, zscale=1))):
        p = W.make_config(cfg, steps=1000, **kw)
        res = run_pair(p, 1000, 32, P.EM_KERNEL_AUTO)
        assert res["E"] < 5e-6 and res["H"] < 1e-5, res


# ------------------------------------------------------- checkpoint / resume, failure detection (include/em.h)
def _full_state(g):
    ck = g.checkpoint()
    return [ck["fields"][c] for c in sorted(ck["fields"])] + [ck["q"]] + ([ck["theta"]] if "theta" in ck else [])


@pytest.mark.parametrize("what", ["leapfrog-fp32", "e-only-fp64", "coupled-fp32", "split-fp64", "coupled-nodal-fp64"])
def test_checkpoint_resume_is_bit_exact_and_check_finite(what):
    """state = fields + q + step index (+ theta): a run interrupted after 5 of 12 steps and resumed in a NEW context
    continues bit for bit (the step index selects the waveform samples; q and theta are accumulators)"""
    precision = 32 if what.endswith("32") else 64
    kw = {}
    p = W.random_problem(37, 29, 23, seed=6100, steps=12, n_ports=5, bc=(0, 1, 0, 0, 1, 0), init_scale=4.0e6 if "coupled" in what else 1.0)
    if what.startswith("e-only"):
        kw["formulation"] = P.EM_FORM_EONLY
    if what.startswith("split"):
        kw["kernel"] = P.EM_KERNEL_SPLIT
    if what.startswith("coupled"):
        th = W.thermal_table(); th[:, 1] *= 2.0e5; th[:, 2] *= 1.0e4
        p.thermal = th
        if "nodal" in what:
            p.thermal_placement = "node"
    ref = P.EM(p, precision=precision, **kw)
    ref.em_step(12)
    a = P.EM(p, precision=precision, **kw)
    a.em_step(5)
    assert a.em_check_finite()
    ck = a.checkpoint()
    assert ck["step"] == 5
    a.close()
    b = P.EM(p, precision=precision, load_init=False, **kw)
    b.resume(ck)
    assert b.step_index == 5
    b.em_step(7)
    for x, y in zip(_full_state(b), _full_state(ref)):
        assert np.array_equal(x, y)
    assert np.abs(_full_state(ref)[-1]).max() > 0
    # failure detection: one NaN in a field, one Inf in q
    bad = ck["fields"][1].copy(); bad[2, 3, 4] = np.nan
    b.em_set_field(1, bad)
    assert not b.em_check_finite()
    b.em_set_field(1, ck["fields"][1])
    assert b.em_check_finite()
    q = ck["q"].copy(); q[0, 0, 0] = np.inf
    b.em_set_joule_energy(q)
    assert not b.em_check_finite()
    with pytest.raises(P.EMError):
        b.em_set_step_index(-1)
    ref.close(); b.close()
