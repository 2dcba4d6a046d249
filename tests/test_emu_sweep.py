"""The product's CUDA sources under CPU emulation (tests/emu) -- memcheck / synccheck / racecheck stand-in, NO GPU needed.

compute-sanitizer is closed on this GPU pool (profiles/r2_sanitizer.md) and, for most of round 2, so was the pool.  These
tests compile paper_2603_07038_b200/csrc/em_lib.cu and its headers, UNMODIFIED, with g++ against an emulation of the CUDA
primitives they use (tests/emu/emu_cuda.h: one fiber per CUDA thread; mbarrier, named-barrier, shuffle and vote
semantics of the PTX ISA; asynchronous TMA / bulk / cp.async copies that complete late and in random order; deadlock
detection; range and alignment checks on every address handed to a copy engine; poisoned shared memory with a canary;
guard pages round the workspace) and then run the SAME parity cases as the `-m gpu` suite -- the test functions of
tests/test_gpu_parity.py, test_gpu_thermal.py and test_gpu_eonly.py are called as they are, with the binding's EM class
swapped for tests/emu/emu_em.EmuEM -- element by element against the oracle.  tests/test_emu_selftest.py shows that
the emulation reports the bugs it is there to catch.

What a green run means: index arithmetic, shared-memory layout, barrier protocol (no CTA barrier in the plane loop),
staging ring reuse, chunk seams, PMC warm-up plane, source cursor and the coupled / E-only / fused-conduction variants
are correct on these grids for every thread schedule tried.  What it does not mean: anything about PTX encodings,
hardware timing or performance -- the C-ABI product has no CPU path and libem.so is never involved here."""
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "emu"))

import workloads as W
from workloads.problem import LOSS_CD, LOSS_EXP
import paper_2603_07038_b200 as P
from oracle import emo
from parity import TOL, compare_state, rel_l2
import build_emu
import emu_em


import test_gpu_parity as TP
import test_gpu_thermal as TT
import test_gpu_eonly as TE
import test_gpu_slabs as TS
import paper_2603_07038_b200.binding as PB

FC = dict(tag="fc", defines=build_emu.VARIANTS["fc"])              # the coupled sweep with the conduction stencil fused in
RACE = dict(tag="race", defines=build_emu.VARIANTS["race"])        # loads / stores instrumented for the racecheck
RACE_FC = dict(tag="race_fc", defines=build_emu.VARIANTS["race_fc"])


def _factory(**fixed):
    def make(p, precision=None, kernel=P.EM_KERNEL_AUTO, device=None, stream=None, lib=None, **kw):
        kw.update(fixed)
        return emu_em.EmuEM(p, precision=precision, kernel=kernel, **kw)
    return make


@pytest.fixture(scope="module", autouse=True)
def _libraries():
    """every library variant used below, compiled side by side if stale (no-op when fresh); only when a test of this
    module actually runs -- collecting the module (e.g. under -m gpu) builds nothing"""
    build_emu.build_all()


@pytest.fixture
def emulated(monkeypatch):
    """P.EM -> EmuEM for the duration of a test; returns a function that switches the library variant"""
    monkeypatch.setenv("EMU_SEED", "0")
    monkeypatch.setattr(P, "EM", _factory())
    monkeypatch.setattr(PB, "EM", _factory())           # (slabs.make_ranks_inprocess takes it from the binding module)

    def variant(**fixed):
        monkeypatch.setattr(P, "EM", _factory(**fixed))
        monkeypatch.setattr(PB, "EM", _factory(**fixed))
    return variant


# ------------------------------------------------------------------------------------------- leapfrog sweep + split
@pytest.mark.parametrize("kernel", [P.EM_KERNEL_SPLIT, P.EM_KERNEL_TMA], ids=["split", "tma"])
@pytest.mark.parametrize("precision", [64, 32])
def test_impulse_example(emulated, kernel, precision):
    TP.test_impulse_example(kernel, precision)


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("dims", TP.SMALL)
def test_random_grids_cd(emulated, dims, precision):
    TP.test_random_grids_cd(dims, precision, P.EM_KERNEL_TMA)


def test_random_grids_cd_split(emulated):
    TP.test_random_grids_cd((37, 29, 23), 64, P.EM_KERNEL_SPLIT)


@pytest.mark.parametrize("zsplit,bc", [(1, (0, 0, 1, 0, 1, 1)), (2, (0,) * 6), (3, (0, 0, 1, 0, 1, 1)), (5, (0,) * 6), (8, (0, 0, 1, 0, 1, 1))])
def test_z_chunks(emulated, zsplit, bc):
    TP.test_tma_sweep_z_chunks(zsplit, bc)


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("dims", [(37, 29, 23), (9, 4, 70)])
def test_random_grids_exp(emulated, dims, precision):
    TP.test_random_grids_exp(dims, precision, P.EM_KERNEL_TMA)


PMC_CASES = [(d, b, pr) for n, (d, b) in enumerate((d, b) for d in [(37, 29, 23), (130, 3, 2), (5, 9, 2), (33, 65, 4)] for b in TP.PMC_BC)
             for pr in ((64, 32) if n % 5 == 0 else (64,) if n % 2 else (32,))]


@pytest.mark.parametrize("dims,bc,precision", PMC_CASES)
def test_random_grids_pmc_walls(emulated, dims, bc, precision):
    TP.test_random_grids_pmc_walls(dims, bc, precision, P.EM_KERNEL_TMA)


def test_pmc_exp_loss_and_z_chunks(emulated):
    TP.test_pmc_exp_loss_and_z_chunks(P.EM_KERNEL_TMA)


def test_percell_ids_pec_material_overlapping_ports(emulated):
    TP.test_random_grid_percell_ids_and_pec_material(P.EM_KERNEL_TMA)
    TP.test_overlapping_ports_add(P.EM_KERNEL_TMA)


def test_api_contract_and_probe(emulated):
    TP.test_api_contract()
    TP.test_probe_matches_fields()


@pytest.mark.parametrize("what", ["leapfrog-fp32", "e-only-fp64", "coupled-fp32", "split-fp64", "coupled-nodal-fp64"])
def test_checkpoint_resume_and_check_finite(emulated, what):
    TP.test_checkpoint_resume_is_bit_exact_and_check_finite(what)


def test_package_slice_several_tiles_and_chunks(emulated):
    """config 4 at 1/8 of the x, y and 1/4 of the z cell counts: 128 x 128 x 48 cells = 2 x 10 tiles, sources, fp32"""
    p = W.make_config(4, scale=8, zscale=4, steps=12)
    TP.run_pair(p, 12, 32, P.EM_KERNEL_TMA, checkpoints=(3,), z_chunks=3)


# -------------------------------------------------------------------------------------------- E-only (eq. (2)) sweep
@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("dims", [(37, 29, 23), (130, 3, 2), (1, 1, 1), (33, 65, 4)])
def test_eonly_random_grids_cd(emulated, dims, precision):
    TE.test_random_grids_cd(dims, precision)


def test_eonly_exp_pmc_chunks(emulated):
    TE.test_random_grids_exp((37, 29, 23), 64)
    TE.test_random_grids_pmc_walls((37, 29, 23), (1, 0, 0, 1, 0, 1), 64)
    TE.test_random_grids_pmc_walls((33, 65, 4), (1, 1, 1, 1, 1, 1), 32)
    TE.test_z_chunks_and_many_ports(3)
    TE.test_percell_ids_pec_material_and_uniform_mu()


def test_eonly_equals_the_leapfrog_kernel(emulated):
    TE.test_equals_the_leapfrog_kernel()


# --------------------------------------------------- coupled sweep (eq. (4)-(6)): conduction kernel + sweep, and fused
VARIANTS = [pytest.param({}, id="k_diffuse+sweep"), pytest.param(FC, id="fused-conduction")]


COUPLED = [pytest.param(d, m, pr, v.values[0], id="%s-%d-fp%d-%s" % ("x".join(map(str, d)), m, pr, v.id))
           for n, (d, m) in enumerate(TT.CASES) for pr in (64, 32) for v in VARIANTS
           if v.values[0] or (n + pr // 32) % 2 == 0]          # fused conduction: every case; conduction kernel: every other one


@pytest.mark.parametrize("dims,mode,precision,variant", COUPLED)
def test_coupled_random_grids(emulated, dims, mode, precision, variant):
    emulated(**variant)
    TT.test_coupled_random_grids(dims, mode, precision, P.EM_KERNEL_AUTO)


@pytest.mark.parametrize("variant", VARIANTS)
def test_coupled_pmc_walls_chunks_diffusion(emulated, variant):
    emulated(**variant)
    TT.test_coupled_with_pmc_walls_and_wall_port(P.EM_KERNEL_AUTO)
    for zsplit in (1, 3, 8):
        TT.test_coupled_sweep_z_chunks(zsplit)
    TT.test_pure_diffusion_and_set_get_temperature()


@pytest.mark.parametrize("variant", VARIANTS)
def test_coupled_package_slice(emulated, variant):
    """the package layout (64 x 64 x 48 cells) with the handbook-order thermal table as it stands, fp32"""
    emulated(**variant)
    p = W.make_config(4, scale=16, zscale=4, steps=16)
    p.thermal = W.thermal_table()
    TT._run(p, 16, 32)


# ------------------------------------------------ nodal thermal stage (theta on the mesh nodes, the paper's placement)
@pytest.mark.parametrize("dims,mode,precision", TT.NODAL_CASES)
def test_nodal_coupled_random_grids(emulated, dims, mode, precision):
    TT.test_nodal_coupled_random_grids(dims, mode, precision)


def test_nodal_pmc_walls_diffusion_api_and_paper_mesh(emulated):
    TT.test_nodal_with_pmc_walls_diffusion_and_api()
    TT.test_nodal_paper_mesh_unknown_count_and_package_slice()


def test_coupled_split_kernels(emulated):
    TT.test_coupled_random_grids((37, 29, 23), LOSS_CD, 64, P.EM_KERNEL_SPLIT)


# ------------------------------------------------------------------ z slabs: pack / unpack kernels and fused peer stores
@pytest.mark.parametrize("n_ranks,mode,precision", [(2, "peer", 32), (3, "peer", 64), (3, "p2p", 32), (2, "p2p", 64)])
def test_slabs_equal_single_domain(emulated, n_ranks, mode, precision):
    """peer mode: the sweep of one slab context stores E'x, E'y straight into the wall plane of the neighbouring
    context's workspace (em_set_peer_halo) -- under the emulation's range checks"""
    TS.test_slabs_equal_single_domain(n_ranks, P.EM_KERNEL_TMA, mode, precision)


@pytest.mark.parametrize("variant", VARIANTS)
def test_thermally_coupled_slabs(emulated, variant):
    emulated(**variant)
    TS.test_thermally_coupled_slabs(P.EM_KERNEL_AUTO, 64)


def test_slabs_split_kernels(emulated):
    TS.test_slabs_equal_single_domain(3, P.EM_KERNEL_SPLIT, "p2p", 32)
    TS.test_thermally_coupled_slabs(P.EM_KERNEL_SPLIT, 64)


@pytest.mark.parametrize("kernel,mode", TS.CASES)
def test_slabs_initial_state_with_pec_material_across_the_cut(emulated, kernel, mode):
    TS.test_slabs_initial_state_with_pec_material_across_the_cut(kernel, mode)


@pytest.mark.parametrize("n_ranks,precision", [(2, 64), (3, 32), (3, 64)])
def test_nodal_thermally_coupled_slabs(emulated, n_ranks, precision):
    TS.test_nodal_thermally_coupled_slabs(n_ranks, precision)


def test_peer_halo_argument_errors(emulated):
    TS.test_peer_halo_argument_errors()


# ---------------------------------------------------------------------------- schedules: every one gives the same bits
def _state(g, thermal):
    out = [g.em_get_field(c) for c in ((0, 1, 2, 3, 4, 5) if g.formulation == P.EM_FORM_LEAPFROG else (0, 1, 2, 6, 7, 8))]
    out.append(g.joule_maps()[1])
    if thermal:
        out.append(g.em_get_temperature_rise())
    return out


SCHEDULE_CASES = [pytest.param(dict(), False, id="leapfrog"), pytest.param(dict(formulation=P.EM_FORM_EONLY), False, id="e-only"),
                  pytest.param(dict(), True, id="coupled"), pytest.param(dict(FC), True, id="coupled-fused-conduction")]


@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("kw,thermal", SCHEDULE_CASES)
def test_random_schedules_do_not_change_a_bit(monkeypatch, kw, thermal, precision):
    """The counterpart of tests/test_gpu_fuzz.py: with EMU_SEED != 0 the fibers run in a random order, whole warps lose
    turns, every synchronisation point may yield and the asynchronous copies complete after random delays and in
    random order.  3 x 4 tiles (fp32) / 5 x 5 (fp64), 3 z chunks, PMC wall at -z (warm-up plane), 40 ports."""
    p = W.random_problem(250, 45, 17, seed=4242, steps=6, n_ports=40, bc=(0, 0, 0, 0, 1, 0), init_scale=4.0e6 if thermal else 1.0)
    if thermal:
        th = W.thermal_table(); th[:, 1] *= 2.0e5; th[:, 2] *= 1.0e4
        p.thermal = th
    ref = None
    for seed in (0, 1, 2, 3):
        monkeypatch.setenv("EMU_SEED", str(seed))
        g = emu_em.EmuEM(p, precision=precision, z_chunks=3, **kw)
        g.em_step(6)
        out = _state(g, thermal)
        g.close()
        if ref is None:
            ref = out
            assert all(np.isfinite(a).all() for a in out) and np.abs(out[0]).max() > 0
        else:
            for a, b in zip(out, ref):
                assert np.array_equal(a, b), seed


# --------------------------------------------------------------- racecheck: no two accesses without an ordering path
@pytest.mark.parametrize("kw,thermal", [pytest.param(dict(RACE), False, id="leapfrog"),
                                        pytest.param(dict(RACE, formulation=P.EM_FORM_EONLY), False, id="e-only"),
                                        pytest.param(dict(RACE), True, id="coupled"),
                                        pytest.param(dict(RACE_FC), True, id="coupled-fused-conduction")])
def test_racecheck_clean(monkeypatch, kw, thermal):
    """EMU_RACECHECK=1 on the -fsanitize=thread build (tests/emu/emu_cuda.h "racecheck"): every load and store of the
    dynamic shared memory is checked against the vector clocks of the barriers; a clean run means that every pair of
    conflicting accesses of k_sweep_tma's barrier-free plane loop is ordered by an mbarrier, a named barrier, a
    __syncwarp or the prologue's __syncthreads -- for ANY schedule, not only the one that ran.  (That the detector and
    this very kernel's barriers are sensitive: tests/test_emu_selftest.py and tests/test_emu_mutations.py.)"""
    monkeypatch.setenv("EMU_RACECHECK", "1")
    monkeypatch.setenv("EMU_SEED", "1")
    p = W.random_problem(130, 31, 9, seed=5, steps=3, n_ports=4, bc=(0, 1, 1, 0, 1, 0), init_scale=4.0e6 if thermal else 1.0)
    if thermal:
        th = W.thermal_table(); th[:, 1] *= 2.0e5; th[:, 2] *= 1.0e4
        p.thermal = th
    g = emu_em.EmuEM(p, precision=32, z_chunks=2, **kw)
    g.em_step(3)                        # (a race would surface as EMError "emu: RACE in kernel ...")
    assert np.isfinite(g.em_get_field(0)).all()
    g.close()


# ------------------------------------------------------------------------------------------- the largest material table
@pytest.mark.parametrize("precision,thermal", [(32, False), (64, False), (32, True), (64, True)])
def test_largest_material_table(emulated, precision, thermal):
    """254 materials + the 'outside / PMC' and 'outside / PEC' entries = the 256-entry table the shared-memory layout must
    hold (em_lib.cu init: the fp64 coupled sweep with its two tables of 32-byte entries does not fit and takes the split
    kernels); ids spread over the whole table"""
    p = W.random_problem(70, 25, 11, seed=77, steps=6, n_ports=3, bc=(1, 0, 0, 1, 0, 1), init_scale=4.0e6 if thermal else 1.0)
    rng = np.random.default_rng(78)
    n = 254
    rep = (n + 15) // 16
    scale = 1.0 + 0.05 * rng.random((rep * 16, 1))
    p.table = (np.tile(np.asarray(p.table, np.float64), (rep, 1)) * scale)[:n]
    p.table[:, 1] = np.tile(np.asarray(p.table[:16, 1]), rep)[:n]                  # (mu unchanged: keeps dt inside the CFL bound)
    p.table[:, 0] = np.maximum(p.table[:, 0], np.tile(np.asarray(p.table[:16, 0]), rep)[:n])
    if getattr(p, "flags", None) is not None:
        p.flags = np.tile(np.asarray(p.flags), rep)[:n]
    p.mat_id = (p.mat_id.astype(np.int64) + 16 * rng.integers(0, rep, size=p.mat_id.shape)).clip(max=n - 1).astype(np.uint8)
    if thermal:
        th = np.tile(W.thermal_table(), (rep, 1))[:n]
        th[:, 1] *= 2.0e5; th[:, 2] *= 1.0e4
        p.thermal = th
        TT._run(p, 6, precision)
    else:
        TP.run_pair(p, 6, precision, P.EM_KERNEL_TMA, z_chunks=2)


# ------------------------------------------------------------------------------------------- random-problem campaign
def _campaign(seed, n_cases, max_cells):
    """random grid shapes (degenerate ones included), walls, loss mode, precision, chunk count, port count, per-cell or
    blocky ids, PEC material, thread schedule -- over the five kernel paths, each case against the oracle"""
    rng = np.random.default_rng(seed)
    done = 0
    while done < n_cases:
        big = rng.random() < 0.3
        nx, ny, nz = int(rng.integers(1, 260 if big else 70)), int(rng.integers(1, 50 if big else 20)), int(rng.integers(1, 24))
        if nx * ny * nz > max_cells:
            continue
        done += 1
        bc = tuple(int(b) for b in (rng.random(6) < 0.35))
        mode, precision = int(rng.integers(0, 2)), int(rng.choice([32, 64]))
        variant = str(rng.choice(["leapfrog", "eonly", "coupled", "fc", "split", "nodal"]))
        zc, nports = int(rng.integers(0, 9)), (int(rng.integers(0, 12)) if nx * ny * nz > 8 else 0)
        # (fp32 + exponential loss: from a RANDOM initial field inside a good conductor the first step cancels E to
        # rounding level there, which the sigma-weighted power map p amplifies beyond 2 tol; from the second step on it
        # does not -- and every configuration of BASELINE.json starts from zero fields or in vacuum)
        steps = int(rng.integers(2 if (mode == 1 and precision == 32) else 1, 9))
        case = dict(dims=(nx, ny, nz), bc=bc, mode=mode, precision=precision, variant=variant, z_chunks=zc, steps=steps, n_ports=nports,
                    seed=int(rng.integers(0, 1 << 30)), emu_seed=int(rng.integers(0, 5)), percell=bool(rng.random() < 0.3), pec=bool(rng.random() < 0.3))
        yield case


def _run_case(case, monkeypatch):
    monkeypatch.setenv("EMU_SEED", str(case["emu_seed"]))
    thermal = case["variant"] in ("coupled", "fc", "nodal")
    if case["variant"] == "eonly" and case["precision"] == 32:
        # the E-only recurrence in fp32 is the one path that is NOT inside north_star's 2e-5 in general (rounding enters the
        # difference of two time levels, gain ~ 1 / (w dt): DESIGN.md section 9 NEXT-4; the long campaign saw 2.8e-5 after 8
        # steps on an 11 x 11 x 3 grid); its fp32 cases run under tests/test_gpu_eonly.py's own bound, the campaign takes fp64
        case = dict(case, precision=64)
    p = W.random_problem(*case["dims"], seed=case["seed"], steps=case["steps"], n_ports=case["n_ports"], loss_mode=case["mode"], bc=case["bc"],
                         blocky=not case["percell"], pec_material=case["pec"], init_scale=4.0e6 if thermal else 1.0)
    kw = dict(z_chunks=case["z_chunks"])
    if thermal:
        th = W.thermal_table(); th[:, 1] *= 2.0e5; th[:, 2] *= 1.0e4
        p.thermal = th
        if case["variant"] == "fc":
            kw.update(FC)
        if case["variant"] == "nodal":
            p.thermal_placement = "node"
    if case["variant"] == "split":
        kw["kernel"] = P.EM_KERNEL_SPLIT
    if case["variant"] == "eonly":
        TE.run_pair(p, case["steps"], case["precision"], z_chunks=case["z_chunks"])
        return
    g = emu_em.EmuEM(p, precision=case["precision"], **kw)
    o = emo.Oracle(p)
    g.em_step(case["steps"]); o.step(case["steps"])
    compare_state(g, o, TOL[case["precision"]])
    if thermal:
        assert rel_l2([g.em_get_temperature_rise()], [o.temperature_rise()]) <= TOL[case["precision"]]
    g.close(); o.close()


def test_random_problem_campaign(emulated, monkeypatch):
    for case in _campaign(20261105, 80, 30000):
        try:
            _run_case(case, monkeypatch)
        except Exception as e:
            raise AssertionError("campaign case %r: %r" % (case, e))


# ---------------------------------------------------------------------------------------- random API-sequence campaign
def _sequence_campaign(seed, n_cases, max_cells):
    """random SEQUENCES of calls on one context -- steps, a field overwritten mid-run (odd and even ping-pong parities), the
    source set replaced, Joule maps read with and without reset, em_reset, the temperature rise overwritten, a checkpoint
    resumed into a second context -- mirrored on the oracle; compared after the sequence and at one point inside it"""
    rng = np.random.default_rng(seed)
    done = 0
    while done < n_cases:
        nx, ny, nz = int(rng.integers(1, 80)), int(rng.integers(1, 20)), int(rng.integers(1, 16))
        if nx * ny * nz > max_cells:
            continue
        done += 1
        variant = str(rng.choice(["leapfrog", "split", "coupled", "fc", "coupled-split", "nodal"]))
        thermal = variant in ("coupled", "fc", "coupled-split", "nodal")
        pec = bool(rng.random() < 0.25)
        kinds = ["step", "step", "step", "set_field", "joule", "joule_reset", "reset", "checkpoint"] + ([] if pec else ["set_source"]) + \
                (["set_theta"] if thermal else [])
        ops = [(str(rng.choice(kinds)), int(rng.integers(0, 1 << 30))) for _ in range(int(rng.integers(3, 9)))] + [("step", int(rng.integers(0, 1 << 30)))]
        yield dict(dims=(nx, ny, nz), bc=tuple(int(b) for b in (rng.random(6) < 0.35)), mode=int(rng.integers(0, 2)), precision=int(rng.choice([32, 64])),
                   variant=variant, z_chunks=int(rng.integers(0, 5)), n_ports=int(rng.integers(0, 10)) if nx * ny * nz > 8 else 0,
                   seed=int(rng.integers(0, 1 << 30)), emu_seed=int(rng.integers(0, 5)), percell=bool(rng.random() < 0.3), pec=pec, ops=ops)


def _run_sequence_case(case, monkeypatch):
    monkeypatch.setenv("EMU_SEED", str(case["emu_seed"]))
    v = case["variant"]
    thermal = v in ("coupled", "fc", "coupled-split", "nodal")
    mk = lambda seed, n_ports: W.random_problem(*case["dims"], seed=seed, steps=64, n_ports=n_ports, loss_mode=case["mode"], bc=case["bc"],
                                                blocky=not case["percell"], pec_material=case["pec"], init_scale=4.0e6 if thermal else 1.0)
    p = mk(case["seed"], case["n_ports"])
    kw = dict(precision=case["precision"], max_ports=32, max_source_edges=1 << 14, max_wave_samples=1 << 14)
    if thermal:
        th = W.thermal_table(); th[:, 1] *= 2.0e5; th[:, 2] *= 1.0e4
        p.thermal = th
        if v == "fc":
            kw.update(FC)
        if v == "nodal":
            p.thermal_placement = "node"
    if v in ("split", "coupled-split"):
        kw["kernel"] = P.EM_KERNEL_SPLIT
    elif v != "nodal":
        kw["z_chunks"] = case["z_chunks"]
    tol = TOL[case["precision"]]
    g = emu_em.EmuEM(p, **kw)
    o = emo.Oracle(p)
    # (fp32 + exponential loss: one step from a random field inside a good conductor is the documented rounding corner of the
    # power map -- DESIGN.md section 9; the sequences take >= 2 steps after every new random field in that combination)
    min_steps = 2 if (case["mode"] == 1 and case["precision"] == 32) else 1
    fresh = True
    src_p = p
    mid = len(case["ops"]) // 2

    def check():
        compare_state(g, o, tol)
        if thermal:
            assert rel_l2([g.em_get_temperature_rise()], [o.temperature_rise()]) <= tol
        # probes = the raw samples of the fields; the layer totals add up to the Joule total; no NaN / Inf
        F = g.fields()
        rp = np.random.default_rng(case["seed"])
        pts = []
        for _ in range(6):
            c = int(rp.integers(0, 6)); sz, sy, sx = g.shapes[c]
            pts.append((c, int(rp.integers(0, sx)), int(rp.integers(0, sy)), int(rp.integers(0, sz))))
        vals, want = g.em_probe(pts), o.probe(pts)
        for v, w, (c, i, j, k) in zip(vals, want, pts):
            assert v == F[c][k, j, i] and abs(v - w) <= tol * max(float(np.max(np.abs(o.get_field(c)))), 1e-300), (c, i, j, k)
        nz = case["dims"][2]; cut = int(rp.integers(0, nz + 1))
        Q = g.joule_maps()[2]
        assert abs(g.em_joule_layers(0, cut) + g.em_joule_layers(cut, nz) - Q) <= 1e-12 * abs(Q)
        assert g.em_check_finite()

    for n, (kind, r) in enumerate(case["ops"]):
        rr = np.random.default_rng(r)
        if kind == "step":
            k = int(rr.integers(min_steps if fresh else 1, 5))
            g.em_step(k); o.step(k); fresh = False
        elif kind == "set_field":
            comp = int(rr.integers(0, 6))
            a = rr.standard_normal(g.shapes[comp]) * (4.0e6 if thermal else 1.0) * (1.0 if comp < 3 else 1.0 / 376.73)
            g.em_set_field(comp, a); o.set_field(comp, a.astype(g.np_dtype).astype(np.float64)); fresh = True
            g.em_step(min_steps); o.step(min_steps); fresh = False
        elif kind == "set_source":
            p2 = mk(int(rr.integers(0, 1 << 30)), int(rr.integers(0, 10)) if p.n_cells > 8 else 0)
            g.em_set_source(p2); o.set_source(p2); src_p = p2
        elif kind in ("joule", "joule_reset"):
            if fresh:
                g.em_step(min_steps); o.step(min_steps); fresh = False
            pg, qg, Qg = g.joule_maps(reset=kind == "joule_reset"); po, qo, Qo = o.joule(reset=kind == "joule_reset")
            assert rel_l2([qg], [qo]) <= tol and rel_l2([pg], [po]) <= 2 * tol and abs(Qg - Qo) <= tol * abs(Qo), (n, kind)
        elif kind == "reset":
            g.em_reset(); o.reset(); fresh = False
        elif kind == "set_theta":
            a = rr.uniform(0.0, 40.0, size=g.theta_shape)
            g.em_set_temperature_rise(a); o.set_temperature_rise(a.astype(g.np_dtype).astype(np.float64))
        elif kind == "checkpoint":                          # carry on in a second context: bit-identical state
            ck = g.checkpoint()
            g2 = emu_em.EmuEM(p, load_init=False, **kw)
            g2.em_set_source(src_p)
            g2.resume(ck)
            for c in range(6):
                assert np.array_equal(g2.em_get_field(c), g.em_get_field(c)), (n, c)
            g.close(); g = g2
        if n == mid and not fresh:
            check()
    check()
    g.close(); o.close()


def test_random_sequence_campaign(emulated, monkeypatch):
    for case in _sequence_campaign(20261107, 40, 12000):
        try:
            _run_sequence_case(case, monkeypatch)
        except Exception as e:
            raise AssertionError("sequence campaign case %r: %r" % (case, e))


@pytest.mark.slow
@pytest.mark.parametrize("seed", [1, 2])
def test_random_sequence_campaign_long(emulated, monkeypatch, seed):
    """EM_RUN_SLOW=1: 2 x 500 sequences (profiles/r2_emulation.md records this round's run)"""
    for case in _sequence_campaign(seed, 500, 30000):
        try:
            _run_sequence_case(case, monkeypatch)
        except Exception as e:
            raise AssertionError("sequence campaign case %r: %r" % (case, e))


def _slab_campaign(seed, n_cases, max_cells):
    """random z-slab decompositions -- grid shape, walls, loss mode, precision, slab count, chunk count, ports, thread
    schedule -- over the transports and the coupled variants; each against the SINGLE-DOMAIN run of the same kernels"""
    rng = np.random.default_rng(seed)
    done = 0
    while done < n_cases:
        nx, ny, nz = int(rng.integers(1, 90)), int(rng.integers(1, 24)), int(rng.integers(4, 20))
        n_ranks = int(rng.integers(2, 5))
        if nx * ny * nz > max_cells or nz < 2 * n_ranks:
            continue
        done += 1
        yield dict(dims=(nx, ny, nz), n_ranks=n_ranks, bc=tuple(int(b) for b in (rng.random(6) < 0.35)), mode=int(rng.integers(0, 2)),
                   precision=int(rng.choice([32, 64])), variant=str(rng.choice(["tma-p2p", "tma-peer", "split-p2p", "coupled", "coupled-split", "nodal"])),
                   z_chunks=int(rng.integers(0, 4)), steps=int(rng.integers(2, 10)), n_ports=int(rng.integers(0, 12)) if nx * ny > 4 else 0,
                   seed=int(rng.integers(0, 1 << 30)), emu_seed=int(rng.integers(0, 5)), percell=bool(rng.random() < 0.3), pec=bool(rng.random() < 0.3))


def _run_slab_case(case, monkeypatch):
    from paper_2603_07038_b200 import slabs
    monkeypatch.setenv("EMU_SEED", str(case["emu_seed"]))
    v = case["variant"]
    thermal = v in ("coupled", "coupled-split", "nodal")
    p = W.random_problem(*case["dims"], seed=case["seed"], steps=case["steps"], n_ports=case["n_ports"], loss_mode=case["mode"], bc=case["bc"],
                         blocky=not case["percell"], pec_material=case["pec"], init_scale=4.0e6 if thermal else 1.0)
    kw = dict(precision=case["precision"])
    if thermal:
        th = W.thermal_table(); th[:, 1] *= 2.0e5; th[:, 2] *= 1.0e4
        p.thermal = th
        if v == "nodal":
            p.thermal_placement = "node"
    if v in ("split-p2p", "coupled-split"):
        kw["kernel"] = P.EM_KERNEL_SPLIT
    elif v != "nodal":
        kw["z_chunks"] = case["z_chunks"]
    ranks = slabs.make_ranks_inprocess(p, case["n_ranks"], mode="peer" if v == "tma-peer" else "p2p", **kw)
    single = emu_em.EmuEM(p, **kw)
    slabs.step_inprocess(ranks, case["steps"]); single.em_step(case["steps"])
    fields, pw, q = slabs.gather_inprocess(ranks)
    fs = single.fields(); ps, qs, Qs = single.joule_maps()
    for c in range(6):
        assert np.array_equal(fields[c], fs[c]), c
    assert np.array_equal(q, qs) and np.array_equal(pw, ps)
    if thermal:
        assert np.array_equal(np.concatenate([r.owned_theta() for r in ranks], axis=0), single.em_get_temperature_rise())
    assert abs(sum(r.joule_total() for r in ranks) - Qs) <= 1e-12 * abs(Qs)
    for r in ranks:
        r.em.close()
    single.close()


def test_random_slab_campaign(emulated, monkeypatch):
    for case in _slab_campaign(20261106, 36, 12000):
        try:
            _run_slab_case(case, monkeypatch)
        except Exception as e:
            raise AssertionError("slab campaign case %r: %r" % (case, e))


@pytest.mark.slow
@pytest.mark.parametrize("seed", [1, 2])
def test_random_slab_campaign_long(emulated, monkeypatch, seed):
    """EM_RUN_SLOW=1: 2 x 600 cases (profiles/r2_emulation.md records this round's run)"""
    for case in _slab_campaign(seed, 600, 30000):
        try:
            _run_slab_case(case, monkeypatch)
        except Exception as e:
            raise AssertionError("slab campaign case %r: %r" % (case, e))


@pytest.mark.slow
@pytest.mark.parametrize("seed", [1, 2, 3, 4])
def test_random_problem_campaign_long(emulated, monkeypatch, seed):
    """EM_RUN_SLOW=1: 4 x 1500 cases (profiles/r2_emulation.md records this round's run)"""
    for case in _campaign(seed, 1500, 60000):
        try:
            _run_case(case, monkeypatch)
        except Exception as e:
            raise AssertionError("campaign case %r: %r" % (case, e))
