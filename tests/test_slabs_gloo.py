"""CPU tests of the z-slab decomposition plumbing (NEXT-3): input slicing, ownership bookkeeping and the
torch.distributed halo exchange (gloo, world_size 2 and 3) with a stand-in context that only stores planes."""
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
    with pytest.raises(ValueError):
        slabs.sub_problem(p, 0, 2)


class _FakeEM:
    """stores Ex / Ey planes only; plane k of rank r holds the value 1000 r + 10 k + comp"""
    def __init__(self, rank, nz, ny=3, nx=4):
        self.shape = {0: (ny + 1, nx), 1: (ny, nx + 1)}
        self.planes = {(c, k): torch.full(self.shape[c], 1000.0 * rank + 10.0 * k + c, dtype=torch.float64)
                       for c in (0, 1) for k in range(nz + 1)}

    def em_get_plane(self, comp, k):
        return self.planes[(comp, k)].clone()

    def em_set_plane(self, comp, k, t):
        assert tuple(t.shape) == self.shape[comp]
        self.planes[(comp, k)] = t.clone()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, nz, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        a, b = slabs.slab_ranges(nz, world)[rank]
        lo, hi = (a - 1 if rank > 0 else 0), (b + 1 if rank < world - 1 else nz)
        sr = slabs.SlabRank(_FakeEM(rank, hi - lo), slabs.SlabMeta(rank, world, a, b, lo, hi, nz))
        slabs.exchange_dist(sr, dist)
        dist.barrier()
        res = {"lo": [sr.em.planes[(c, 0)][0, 0].item() for c in (0, 1)],
               "hi": [sr.em.planes[(c, hi - lo)][0, 0].item() for c in (0, 1)], "a": a, "b": b, "lo_": lo, "hi_": hi}
        torch.save(res, os.path.join(out, "r%d.pt" % rank))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_exchange_dist_gloo(world, tmp_path):
    nz = 13
    mp.spawn(_worker, args=(world, _free_port(), nz, str(tmp_path)), nprocs=world, join=True)
    res = [torch.load(os.path.join(str(tmp_path), "r%d.pt" % r)) for r in range(world)]
    for r in range(world):
        me = res[r]
        if r > 0:            # my lower wall plane <- the lower neighbour's global node plane b_low - 1 = a - 1
            nb = res[r - 1]
            k_local = (nb["b"] - 1) - nb["lo_"]
            assert me["lo"] == [1000.0 * (r - 1) + 10.0 * k_local + c for c in (0, 1)]
        else:                # a real wall keeps its own values
            assert me["lo"] == [0.0, 1.0]
        if r < world - 1:    # my upper wall plane <- the upper neighbour's global node plane a_up + 1 = b + 1
            nb = res[r + 1]
            k_local = (nb["a"] + 1) - nb["lo_"]
            assert me["hi"] == [1000.0 * (r + 1) + 10.0 * k_local + c for c in (0, 1)]
        else:
            assert me["hi"] == [1000.0 * r + 10.0 * (me["hi_"] - me["lo_"]) + c for c in (0, 1)]
