"""CPU tests of the z-slab decomposition plumbing (NEXT-3): input slicing, ownership bookkeeping and the
torch.distributed halo exchange (gloo, world_size 2 and 3) around a NumPy stand-in context that runs a real recurrence
with the data dependencies of the sweep (its single-domain run is the closed form the slabs must reproduce)."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as W
from paper_2603_07038_b200 import slabs


def test_ranges_and_sub_problem_slicing():
    assert slabs.slab_ranges(13, 3) == [(0, 4), (4, 8), (8, 13)]
    with pytest.raises(ValueError):
        slabs.slab_ranges(5, 3)
    p = W.random_problem(6, 5, 13, seed=1, n_ports=30, steps=5, bc=(0, 1, 0, 0, 0, 0))
    metas = []
    for r in range(3):
        s, m = slabs.sub_problem(p, r, 3)
        metas.append(m)
        assert (m.lo, m.hi) == ((0, 5), (3, 9), (7, 13))[r]
        assert s.nz == m.hi - m.lo and s.mat_id.shape == (s.nz, 5, 6)
        assert np.array_equal(s.dz, p.dz[m.lo:m.hi]) and np.array_equal(s.mat_id, p.mat_id[m.lo:m.hi])
        assert s.bc == ((0, 1, 0, 0, 0, 1), (0, 1, 0, 0, 1, 1), (0, 1, 0, 0, 1, 0))[r]      # PMC on artificial walls only
        assert s.init[0].shape == (s.nz + 1, 6, 6) and s.init[2].shape == (s.nz, 6, 7)
        assert np.array_equal(s.init[5], p.init[5][m.lo:m.hi + 1])
        assert s.n_ports == p.n_ports
        # every kept edge is the original edge shifted by lo, and every original edge inside the slab is kept
        kept = {(int(c), int(i), int(j), int(k) + m.lo) for c, (i, j, k) in zip(s.edge_comp, s.edge_ijk)}
        want = {(int(c), int(i), int(j), int(k)) for c, (i, j, k) in zip(p.edge_comp, p.edge_ijk)
                if m.lo <= k <= (m.hi if c != 2 else m.hi - 1)}
        assert kept == want
    # owned layers tile [0, nz) exactly
    assert [(m.a, m.b) for m in metas] == [(0, 4), (4, 8), (8, 13)]
    p.thermal = W.thermal_table()
    s, m = slabs.sub_problem(p, 1, 3)                            # the coupled problem shards too (theta rides in the halo)
    assert s.thermal is p.thermal


class _StandInEM:
    """A NumPy stand-in for the library with the halo calls of include/em.h and a REAL recurrence with the data
    dependencies of the sweep: node planes u[k] (Ex and Ey stacks) advance by a 3-point stencil in z, cell layers (theta)
    by a 3-point diffusion; a real wall plane is held (Dirichlet), a real end layer reflects; an ARTIFICIAL wall plane and
    a ghost layer compute garbage that only the halo exchange can repair.  The single-domain run of the same class is
    the closed form the assembled slabs must reproduce bit for bit."""
    C1, C2 = 0.23, 0.11

    def __init__(self, u_ex, u_ey, theta, wall_lo_real=True, wall_hi_real=True):
        self.ex, self.ey, self.th = u_ex.copy(), u_ey.copy(), theta.copy()
        self.real = (wall_lo_real, wall_hi_real)
        self.nz = theta.shape[0]
        self.n0, self.n1, self.n2 = self.ex[0].size, self.ey[0].size, self.th[0].size
        self.device = "cpu"

    def new_halo_buffer(self):
        return torch.empty(self.n0 + self.n1 + self.n2, dtype=torch.float64)

    def em_step(self, n=1):
        for _ in range(n):
            for u in (self.ex, self.ey):
                new = u.copy()
                new[1:-1] = u[1:-1] + self.C1 * (u[2:] - 2.0 * u[1:-1] + u[:-2])
                if not self.real[0]:
                    new[0] = 0.5 * u[0] + 7.0                      # garbage on an artificial wall
                if not self.real[1]:
                    new[-1] = -3.0 * u[-1] - 1.0
                u[...] = new
            t = self.th
            lo = np.concatenate([t[:1], t[:-1]]); hi = np.concatenate([t[1:], t[-1:]])     # reflecting ends
            new = t + self.C2 * (hi - 2.0 * t + lo)
            if not self.real[0]:
                new[0] = 1.0e3                                      # garbage in a ghost layer
            if not self.real[1]:
                new[-1] = -1.0e3
            t[...] = new

    def em_get_halo(self, kp, kl, out, stream=None):
        out[:self.n0] = torch.from_numpy(self.ex[kp].ravel()); out[self.n0:self.n0 + self.n1] = torch.from_numpy(self.ey[kp].ravel())
        out[self.n0 + self.n1:] = torch.from_numpy(self.th[kl].ravel())
        return out

    def em_set_halo(self, kp, kl, src, stream=None):
        a = src.numpy()
        self.ex[kp] = a[:self.n0].reshape(self.ex[kp].shape); self.ey[kp] = a[self.n0:self.n0 + self.n1].reshape(self.ey[kp].shape)
        self.th[kl] = a[self.n0 + self.n1:].reshape(self.th[kl].shape)

    def em_joule_layers(self, k0, k1):
        return float(self.th[k0:k1].sum())


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _global_state(nz, ny=3, nx=4, seed=5):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((nz + 1, ny + 1, nx)), rng.standard_normal((nz + 1, ny, nx + 1)), rng.standard_normal((nz, ny, nx))


def _worker(rank, world, port, nz, steps, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        m = slabs.slab_meta(nz, rank, world)
        ex, ey, th = _global_state(nz)
        em = _StandInEM(ex[m.lo:m.hi + 1], ey[m.lo:m.hi + 1], th[m.lo:m.hi], not m.has_below, not m.has_above)
        sr = slabs.SlabRank(em, m)
        sr.step(steps, dist)
        total = sr.joule_total(dist)
        k0, k1 = m.a - m.lo, m.b - m.lo
        last = 1 if not m.has_above else 0
        np.savez(os.path.join(out, "r%d.npz" % rank), ex=em.ex[k0:k1 + last], ey=em.ey[k0:k1 + last], th=em.th[k0:k1], total=total)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_exchange_dist_gloo_reproduces_the_single_domain_recurrence(world, tmp_path):
    nz, steps = 13, 25
    mp.spawn(_worker, args=(world, _free_port(), nz, steps, str(tmp_path)), nprocs=world, join=True)
    ex, ey, th = _global_state(nz)
    ref = _StandInEM(ex, ey, th)
    ref.em_step(steps)
    parts = [np.load(os.path.join(str(tmp_path), "r%d.npz" % r)) for r in range(world)]
    assert np.array_equal(np.concatenate([p["ex"] for p in parts]), ref.ex)
    assert np.array_equal(np.concatenate([p["ey"] for p in parts]), ref.ey)
    assert np.array_equal(np.concatenate([p["th"] for p in parts]), ref.th)
    # the all-reduced total of the owned layers is the single-domain total on every rank
    for p in parts:
        assert abs(float(p["total"]) - ref.th.sum()) <= 1e-12 * abs(ref.th).sum()
    assert np.abs(ref.ex - ex).max() > 1e-3                      # the recurrence did something


class _WiringEM:
    """records what the peer wiring hands to em_set_peer_halo (no CUDA involved)"""
    def __init__(self, rank):
        self.workspace_ptr = 0x10000000 * (rank + 1)
        self.rank = rank
        self.calls = []

    def wall_offsets(self, side):               # [parity * 2 + comp], distinct per rank and side
        return [1000 * self.rank + 100 * side + 10 * q + c for q in (0, 1) for c in (0, 1)]

    def em_set_peer_halo(self, side, k_send, addresses):
        self.calls.append((side, k_send, list(addresses)))


def test_peer_wiring_hands_each_sweep_its_neighbours_wall_planes():
    """in-process peer wiring (slabs.connect_peers_inprocess): rank r stores its plane b-1 into the -z wall of rank r+1 and
    its plane a+1 into the +z wall of rank r-1; the addresses are the neighbour's workspace base + ITS wall offsets"""
    nz, world = 13, 3
    ranks = [slabs.SlabRank(_WiringEM(r), slabs.slab_meta(nz, r, world)) for r in range(world)]
    slabs.connect_peers_inprocess(ranks)
    for r, sr in enumerate(ranks):
        m = sr.meta
        want = []
        if m.has_above:
            nb = ranks[r + 1].em
            want.append((1, m.b - 1 - m.lo, [nb.workspace_ptr + o for o in nb.wall_offsets(0)]))
        if m.has_below:
            nb = ranks[r - 1].em
            want.append((0, m.a + 1 - m.lo, [nb.workspace_ptr + o for o in nb.wall_offsets(1)]))
        assert sr.em.calls == want and sr.mode == "peer"
    # the plane a slab sends up is the plane its upper neighbour holds as wall plane 0, and vice versa (global indices)
    for r in range(world - 1):
        lo, hi = ranks[r], ranks[r + 1]
        assert lo.meta.lo + lo.k_send_up == hi.meta.lo + hi.k_wall_lo
        assert hi.meta.lo + hi.k_send_down == lo.meta.lo + lo.k_wall_hi
        assert lo.meta.lo + lo.layer_send_up == hi.meta.lo + 0                       # theta: my top owned layer = its ghost layer 0
        assert hi.meta.lo + hi.layer_send_down == lo.meta.lo + lo.nz_local - 1       # my bottom owned layer = its last ghost layer


# ---- the REAL kernels under the exchange, one process per slab, gloo: the product's sweep sources on the emulated build ----
# (tests/emu: em_lib.cu compiled against the CPU emulation of the CUDA primitives; no GPU.  This is the N > 1 path of
# bench.py --gpus N --decomp slabs with transport p2p -- sub_problem, SlabRank.step, exchange_dist with the pack / unpack
# kernels, the all-reduced Joule total -- with every arithmetic step in the kernels' own code.)
def _problem_for_slabs(thermal):
    p = W.random_problem(21, 18, 13, seed=9400, steps=12, n_ports=25, bc=(0, 1, 0, 0, 0, 1), init_scale=4.0e6 if thermal else 1.0)
    if thermal:
        th = W.thermal_table(); th[:, 1] *= 2.0e5; th[:, 2] *= 1.0e4
        p.thermal = th
        if thermal == "node":
            p.thermal_placement = "node"                  # theta on the mesh nodes: the halo carries a node plane of it
    return p


def _emu_worker(rank, world, port, thermal, steps, out):
    sys.path.insert(0, os.path.join(ROOT, "tests", "emu"))
    import emu_em
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), EMU_THREADS="2")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        s, meta = slabs.sub_problem(_problem_for_slabs(thermal), rank, world)
        sr = slabs.SlabRank(emu_em.EmuEM(s, precision=64), meta, mode="p2p")
        sr.step(steps, dist)
        total = sr.joule_total(dist)
        fields = sr.owned_fields()
        extra = {"theta": sr.owned_theta()} if thermal else {}
        np.savez(os.path.join(out, "r%d.npz" % rank), total=total, q=sr.owned_joule()[1], **{"f%d" % c: f for c, f in enumerate(fields)}, **extra)
        dist.barrier()
        sr.em.close()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,thermal", [(2, False), (3, True), (2, "node")])
def test_real_kernels_under_the_gloo_exchange_equal_the_single_domain_run(world, thermal, tmp_path):
    sys.path.insert(0, os.path.join(ROOT, "tests", "emu"))
    import build_emu
    import emu_em
    build_emu.build_emu()                      # (before the workers start: they must not race to build it)
    steps = 12
    mp.spawn(_emu_worker, args=(world, _free_port(), thermal, steps, str(tmp_path)), nprocs=world, join=True)
    p = _problem_for_slabs(thermal)
    single = emu_em.EmuEM(p, precision=64)
    single.em_step(steps)
    fs = single.fields(); _, qs, Qs = single.joule_maps()
    parts = [np.load(os.path.join(str(tmp_path), "r%d.npz" % r)) for r in range(world)]
    for c in range(6):
        assert np.array_equal(np.concatenate([pt["f%d" % c] for pt in parts], axis=0), fs[c]), c      # bit for bit
    assert np.array_equal(np.concatenate([pt["q"] for pt in parts], axis=0), qs)
    if thermal:
        assert np.array_equal(np.concatenate([pt["theta"] for pt in parts], axis=0), single.em_get_temperature_rise())
    for pt in parts:                                                                                     # all-reduced on every rank
        assert abs(float(pt["total"]) - Qs) <= 1e-12 * abs(Qs) and Qs > 0
    single.close()
