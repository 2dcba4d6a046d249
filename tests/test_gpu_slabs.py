"""z-slab decomposition (NEXT-3) on ONE GPU: the slab contexts run one after another and exchange
their halos either with the pack / unpack kernels (mode "p2p") or by the stores fused into the sweep (mode "peer");
the assembled result must equal the single-domain run of the same library BIT FOR BIT (itself parity-checked against
the oracle) and match the oracle.  The last test wires two PROCESSES sharing the GPU through CUDA IPC."""
import os
import socket
import sys

import numpy as np
import pytest

import workloads as W
from workloads.problem import LOSS_CD, LOSS_EXP
import paper_2603_07038_b200 as P
from paper_2603_07038_b200 import slabs
from oracle import emo
from parity import rel_l2, TOL

pytestmark = pytest.mark.gpu

CASES = [pytest.param(P.EM_KERNEL_TMA, "p2p", id="tma-p2p"), pytest.param(P.EM_KERNEL_TMA, "peer", id="tma-peer"),
         pytest.param(P.EM_KERNEL_SPLIT, "p2p", id="split-p2p")]


@pytest.mark.parametrize("n_ranks", [2, 3])
@pytest.mark.parametrize("kernel,mode", CASES)
@pytest.mark.parametrize("precision", [64, 32])
def test_slabs_equal_single_domain(n_ranks, kernel, mode, precision):
    p = W.random_problem(21, 18, 13, seed=9000 + n_ranks, loss_mode=LOSS_CD, steps=40, n_ports=25, bc=(0, 1, 0, 0, 0, 1))
    ranks = slabs.make_ranks_inprocess(p, n_ranks, mode=mode, precision=precision, kernel=kernel)
    single = P.EM(p, precision=precision, kernel=kernel)
    o = emo.Oracle(p)
    slabs.step_inprocess(ranks, 40); single.em_step(40); o.step(40)
    fields, pw, q = slabs.gather_inprocess(ranks)
    fs = single.fields(); ps, qs, Qs = single.joule_maps()
    # same kernels, same inputs plane by plane: identical bits
    for c in range(6):
        assert fields[c].shape == fs[c].shape
        assert np.array_equal(fields[c], fs[c]), c
    assert np.array_equal(q, qs) and np.array_equal(pw, ps)
    fo = o.fields(); _, qo, Qo = o.joule()
    tol = TOL[precision]
    assert rel_l2(fields[:3], fo[:3]) <= tol and rel_l2(fields[3:], fo[3:]) <= tol and rel_l2([q], [qo]) <= tol
    # the Joule total of the problem = the sum of the owned layers' totals (the all-reduce of SURVEY.md 8(e))
    Q = sum(r.joule_total() for r in ranks)
    assert abs(Q - Qo) <= tol * Qo and abs(Q - Qs) <= 1e-12 * Qs
    for r in ranks:
        r.em.close()
    single.close(); o.close()


@pytest.mark.parametrize("kernel,mode", CASES)
def test_slabs_initial_state_with_pec_material_across_the_cut(kernel, mode):
    """an initial Ex, Ey on a slab's wall plane whose edge touches a PEC-flagged cell ABOVE the plane (a cell the slab does
    not hold) is forced to 0 in the single-domain run; the slab learns it from its neighbour in the exchange that precedes
    the first step (slabs.SlabRank.halo_synced).  The case is the one the random slab campaign of tests/test_emu_sweep.py found."""
    p = W.random_problem(62, 23, 7, seed=811118369, loss_mode=LOSS_EXP, steps=2, n_ports=8, blocky=False, pec_material=True)
    ranks = slabs.make_ranks_inprocess(p, 3, mode=mode, precision=32, kernel=kernel)
    single = P.EM(p, precision=32, kernel=kernel)
    slabs.step_inprocess(ranks, 2); single.em_step(2)
    fields, pw, q = slabs.gather_inprocess(ranks)
    fs = single.fields(); ps, qs, _ = single.joule_maps()
    assert any(np.any(f != 0) for f in fs)
    for c in range(6):
        assert np.array_equal(fields[c], fs[c]), c
    assert np.array_equal(q, qs) and np.array_equal(pw, ps)
    for r in ranks:
        r.em.close()
    single.close()


@pytest.mark.parametrize("mode", ["p2p", "peer"])
def test_slabs_config4_scaled_ports_everywhere(mode):
    p = W.make_config(4, scale=16, zscale=4, steps=60)            # 64 x 64 x 48, ports in several layers
    ranks = slabs.make_ranks_inprocess(p, 4, mode=mode, precision=32, z_chunks=2)
    o = emo.Oracle(p)
    slabs.step_inprocess(ranks, 60); o.step(60)
    fields, pw, q = slabs.gather_inprocess(ranks)
    fo = o.fields(); _, qo, _ = o.joule()
    assert rel_l2(fields[:3], fo[:3]) <= 2e-5 and rel_l2(fields[3:], fo[3:]) <= 2e-5 and rel_l2([q], [qo]) <= 2e-5
    for r in ranks:
        r.em.close()


@pytest.mark.parametrize("kernel", [P.EM_KERNEL_AUTO, P.EM_KERNEL_SPLIT])
@pytest.mark.parametrize("precision", [64, 32])
def test_thermally_coupled_slabs(kernel, precision):
    """the coupled step shards too: the halo carries the temperature rise of the owned boundary layer into the
    neighbour's ghost layer (theta and sigma(T) there feed the owned layer's conduction and edge conductivities)"""
    p = W.random_problem(21, 18, 14, seed=9100, loss_mode=LOSS_CD, steps=40, n_ports=20, init_scale=4.0e6)
    th = W.thermal_table(); th[:, 1] *= 2.0e5; th[:, 2] *= 1.0e4      # conduction and TCR exaggerated (test_gpu_thermal.py)
    p.thermal = th
    ranks = slabs.make_ranks_inprocess(p, 3, precision=precision, kernel=kernel)
    single = P.EM(p, precision=precision, kernel=kernel)
    o = emo.Oracle(p)
    slabs.step_inprocess(ranks, 40); single.em_step(40); o.step(40)
    fields, pw, q = slabs.gather_inprocess(ranks)
    theta = np.concatenate([r.owned_theta() for r in ranks], axis=0)
    fs = single.fields(); _, qs, _ = single.joule_maps(); ts = single.em_get_temperature_rise()
    for c in range(6):
        assert np.array_equal(fields[c], fs[c]), c
    assert np.array_equal(q, qs) and np.array_equal(theta, ts)
    to = o.temperature_rise()
    assert np.max(np.abs(to)) > 0 and rel_l2([theta], [to]) <= TOL[precision]
    assert rel_l2(fields[:3], o.fields()[:3]) <= TOL[precision]
    for r in ranks:
        r.em.close()
    single.close(); o.close()


@pytest.mark.parametrize("n_ranks", [2, 3])
@pytest.mark.parametrize("precision", [64, 32])
def test_nodal_thermally_coupled_slabs(n_ranks, precision):
    """the paper's placement (theta on the mesh nodes, em_grid.thermal = EM_THERMAL_NODE) shards the same way: the halo
    carries the temperature rise of the node plane that carries Ex, Ey -- a slab cannot update the nodes of its artificial
    wall plane (half of their cells, edges and heat lie in the neighbour) -- and sigma(T) of the ghost layer follows"""
    p = W.random_problem(17, 14, 13, seed=9150 + n_ranks, loss_mode=LOSS_CD if n_ranks == 2 else LOSS_EXP, steps=40, n_ports=12,
                         init_scale=4.0e6, bc=(0, 1, 0, 0, 1, 0))
    th = W.thermal_table(); th[:, 1] *= 2.0e5; th[:, 2] *= 1.0e4
    p.thermal = th
    p.thermal_placement = "node"
    ranks = slabs.make_ranks_inprocess(p, n_ranks, precision=precision)
    single = P.EM(p, precision=precision)
    o = emo.Oracle(p)
    slabs.step_inprocess(ranks, 40); single.em_step(40); o.step(40)
    fields, pw, q = slabs.gather_inprocess(ranks)
    theta = np.concatenate([r.owned_theta() for r in ranks], axis=0)
    fs = single.fields(); _, qs, Qs = single.joule_maps(); ts = single.em_get_temperature_rise()
    assert theta.shape == ts.shape == (p.nz + 1, p.ny + 1, p.nx + 1)
    for c in range(6):
        assert np.array_equal(fields[c], fs[c]), c
    assert np.array_equal(q, qs) and np.array_equal(theta, ts)
    to = o.temperature_rise()
    assert np.max(np.abs(p.thermal[p.mat_id, 2])) * np.max(to) > 1e-3             # the feedback on sigma matters
    assert rel_l2([theta], [to]) <= TOL[precision] and rel_l2(fields[:3], o.fields()[:3]) <= TOL[precision]
    Q = sum(r.joule_total() for r in ranks)
    assert abs(Q - Qs) <= 1e-12 * Qs and abs(Q - o.joule()[2]) <= TOL[precision] * Qs
    for r in ranks:
        r.em.close()
    single.close(); o.close()


def test_peer_halo_argument_errors():
    p = W.random_problem(9, 8, 7, seed=9200, n_ports=0)
    g = P.EM(p, precision=64)
    with pytest.raises(P.EMError) as e:
        g.em_set_peer_halo(1, 3, [g.workspace_ptr] * 4)           # the +z wall of this context is a real PEC wall
    assert e.value.code == 4
    with pytest.raises(P.EMError):
        g.em_wall_offset(2, 0, 0)
    eo = P.EM(p, precision=64, formulation=P.EM_FORM_EONLY)
    with pytest.raises(P.EMError) as e:
        eo.em_get_halo(1, 0, eo._torch.empty(1000, dtype=eo.dtype, device=eo.device))
    assert e.value.code == 5
    g.close(); eo.close()
    s, _ = slabs.sub_problem(W.random_problem(9, 8, 7, seed=9201, n_ports=0), 0, 2)      # a slab with an artificial +z wall
    gs = P.EM(s, precision=64)
    with pytest.raises(P.EMError) as e:
        gs.em_set_peer_halo(1, 2, [gs.workspace_ptr + 8] * 4)      # the sweep stores 16 bytes at a time
    assert e.value.code == 1
    gs.em_set_peer_halo(1, 2, [gs.workspace_ptr] * 4)
    gs.em_set_peer_halo(1, 0, None)
    gs.close()


# ---- two processes sharing the GPU: CUDA IPC peer mapping + gloo for the host-side barrier ----------------------------
def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _ipc_worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        torch.cuda.set_device(0)
        p = W.random_problem(21, 18, 13, seed=9300, loss_mode=LOSS_CD, steps=30, n_ports=25, bc=(0, 1, 0, 0, 0, 1))
        s, meta = slabs.sub_problem(p, rank, world)
        sr = slabs.SlabRank(P.EM(s, precision=64), meta)
        slabs.connect_peers_dist(sr, dist)
        sr.step(30, dist)
        torch.cuda.synchronize()
        Q = sr.joule_total(dist)
        np.savez(os.path.join(out_dir, "r%d.npz" % rank), Q=Q, **{"f%d" % c: f for c, f in enumerate(sr.owned_fields())})
        dist.barrier()
        sr.em.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.slow          # two processes on ONE GPU: opt-in (EM_RUN_SLOW=1); it passed in the three full-suite runs of round 2
def test_peer_halo_between_two_processes_over_cuda_ipc(tmp_path):
    import torch.multiprocessing as mp
    world = 2
    mp.spawn(_ipc_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    p = W.random_problem(21, 18, 13, seed=9300, loss_mode=LOSS_CD, steps=30, n_ports=25, bc=(0, 1, 0, 0, 0, 1))
    single = P.EM(p, precision=64)
    single.em_step(30)
    fs = single.fields(); Qs = single.em_joule(None, None, total=True)
    parts = [np.load(os.path.join(str(tmp_path), "r%d.npz" % r)) for r in range(world)]
    for c in range(6):
        assert np.array_equal(np.concatenate([pt["f%d" % c] for pt in parts], axis=0), fs[c]), c
    assert all(abs(float(pt["Q"]) - Qs) <= 1e-12 * Qs for pt in parts)
    single.close()
