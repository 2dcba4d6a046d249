"""z-slab decomposition of the EM time-marching over several GPUs (NEXT-3 of SURVEY.md 8(f)).

One process per GPU, each with its own em_ctx over its slab of cell layers [a, b) EXTENDED by one ghost cell layer on
every interior side.  The artificial end walls of the extended slab are PMC walls (include/em.h EM_BC_PMC): their
tangential E (Ex, Ey on the wall's node plane) is an unknown that the library lets the caller overwrite, and it is
the ONLY thing a slab cannot compute itself -- everything one plane inside the wall (H', E'z of the ghost layer, the
Joule sum that closes on the plane above) follows from correct inputs.  So the exchange after every step is
    to the slab above : my Ex, Ey at global node plane b-1   -> its lower wall plane
    to the slab below : my Ex, Ey at global node plane a+1   -> its upper wall plane
i.e. two planes per neighbour per step (2 x nx*ny reals), point-to-point only.  All arithmetic stays
in the CUDA kernels; this module only slices inputs (host) and moves planes (em_get_plane / em_set_plane + send/recv).

The path of BASELINE.json is one GPU; this is the multi-GPU scale-out of the same kernels, tested on one GPU by running
the slab contexts one after another (no kernel waits on another) and, for the exchange logic, with gloo on CPU.
"""
from __future__ import annotations

import copy
import dataclasses
from typing import List, Sequence

import numpy as np

BC_PMC = 1


@dataclasses.dataclass
class SlabMeta:
    rank: int
    n_ranks: int
    a: int          # first owned cell layer (global)
    b: int          # one past the last owned cell layer
    lo: int         # first cell layer of the extended slab (a - 1 on interior sides)
    hi: int         # one past the last cell layer of the extended slab (b + 1 on interior sides)
    nz: int         # global nz

    @property
    def has_below(self) -> bool:
        return self.rank > 0

    @property
    def has_above(self) -> bool:
        return self.rank < self.n_ranks - 1


def slab_ranges(nz: int, n_ranks: int):
    """balanced owned ranges [a, b) of cell layers; every slab needs >= 2 layers"""
    if n_ranks < 1 or nz < 2 * n_ranks:
        raise ValueError("need at least 2 cell layers per slab")
    cuts = [(nz * r) // n_ranks for r in range(n_ranks + 1)]
    return [(cuts[r], cuts[r + 1]) for r in range(n_ranks)]


def sub_problem(p, rank: int, n_ranks: int):
    """The inputs of slab `rank`: a shallow copy of the problem restricted to the extended slab, with PMC on the
    artificial walls, the port edges that fall inside it (k shifted) and the matching slices of the initial fields."""
    if getattr(p, "thermal", None) is not None:
        raise ValueError("the slab decomposition covers the EM + Joule path; thermal conduction needs a theta halo")
    a, b = slab_ranges(p.nz, n_ranks)[rank]
    lo = a - 1 if rank > 0 else 0
    hi = b + 1 if rank < n_ranks - 1 else p.nz
    meta = SlabMeta(rank, n_ranks, a, b, lo, hi, p.nz)
    s = copy.copy(p)
    s.name = "%s_slab%d_of_%d" % (p.name, rank, n_ranks)
    s.nz = hi - lo
    s.dz = np.ascontiguousarray(p.dz[lo:hi])
    s.mat_id = np.ascontiguousarray(p.mat_id[lo:hi])
    bc = list(getattr(p, "bc", (0,) * 6))
    if meta.has_below:
        bc[4] = BC_PMC
    if meta.has_above:
        bc[5] = BC_PMC
    s.bc = tuple(bc)
    # ports: keep every port (same waveform table and indices), keep the edges inside the extended slab
    comp, ijk, wt, beg, end = [], [], [], [], []
    for q in range(p.n_ports):
        beg.append(len(comp))
        for e in range(int(p.port_edge_begin[q]), int(p.port_edge_end[q])):
            c = int(p.edge_comp[e]); i, j, k = (int(v) for v in p.edge_ijk[e])
            top = hi if c != 2 else hi - 1                   # Ex, Ey live on node planes lo..hi; Ez on layers lo..hi-1
            if lo <= k <= top:
                comp.append(c); ijk.append((i, j, k - lo)); wt.append(float(p.edge_weight[e]))
        end.append(len(comp))
    s.port_edge_begin = np.asarray(beg, np.int64); s.port_edge_end = np.asarray(end, np.int64)
    s.edge_comp = np.asarray(comp, np.int32); s.edge_ijk = np.asarray(ijk, np.int32).reshape(-1, 3)
    s.edge_weight = np.asarray(wt, np.float64)
    if getattr(p, "init", None):
        node = (0, 1, 5)                                     # Ex, Ey, Hz: nz + 1 planes; Ez, Hx, Hy: nz layers
        s.init = {c: np.ascontiguousarray(f[lo:hi + 1] if c in node else f[lo:hi]) for c, f in p.init.items()}
    s.probes = np.zeros((0, 4), np.int32)
    return s, meta


class SlabRank:
    """One slab: its context (anything with em_step / em_get_plane / em_set_plane / em_get_field / joule_maps) and
    the plane bookkeeping of the exchange."""

    def __init__(self, em, meta: SlabMeta):
        self.em, self.meta = em, meta

    # local plane indices ------------------------------------------------------------------------------------
    @property
    def k_send_up(self) -> int:        # global node plane b - 1
        return self.meta.b - 1 - self.meta.lo

    @property
    def k_send_down(self) -> int:      # global node plane a + 1
        return self.meta.a + 1 - self.meta.lo

    @property
    def k_wall_lo(self) -> int:
        return 0

    @property
    def k_wall_hi(self) -> int:
        return self.meta.hi - self.meta.lo

    def planes_up(self):
        return [self.em.em_get_plane(0, self.k_send_up), self.em.em_get_plane(1, self.k_send_up)]

    def planes_down(self):
        return [self.em.em_get_plane(0, self.k_send_down), self.em.em_get_plane(1, self.k_send_down)]

    def set_wall_lo(self, planes):
        self.em.em_set_plane(0, self.k_wall_lo, planes[0]); self.em.em_set_plane(1, self.k_wall_lo, planes[1])

    def set_wall_hi(self, planes):
        self.em.em_set_plane(0, self.k_wall_hi, planes[0]); self.em.em_set_plane(1, self.k_wall_hi, planes[1])

    # owned parts of the results (NumPy, global k order) ---------------------------------------------------------
    def owned_fields(self):
        m = self.meta
        last = not m.has_above
        out = []
        for c in range(6):
            f = self.em.em_get_field(c)
            node = c in (0, 1, 5)
            k0 = m.a - m.lo
            k1 = m.b - m.lo + (1 if (node and last) else 0)     # the last slab also owns node plane nz
            out.append(f[k0:k1])
        return out

    def owned_joule(self):
        m = self.meta
        pw, q, _ = self.em.joule_maps()
        return pw[m.a - m.lo:m.b - m.lo], q[m.a - m.lo:m.b - m.lo]


def exchange_inprocess(ranks: Sequence[SlabRank]):
    """Halo exchange between slab contexts that live in ONE process (one GPU, run one after another): plain device
    copies through em_get_plane / em_set_plane.  Used by the single-GPU tests of the decomposition."""
    ups = [r.planes_up() if r.meta.has_above else None for r in ranks]
    downs = [r.planes_down() if r.meta.has_below else None for r in ranks]
    for n, r in enumerate(ranks):
        if r.meta.has_below:
            r.set_wall_lo(ups[n - 1])
        if r.meta.has_above:
            r.set_wall_hi(downs[n + 1])


def _pack(planes):
    import torch
    return torch.cat([planes[0].reshape(-1), planes[1].reshape(-1)])


def _unpack(buf, like):
    n0 = like[0].numel()
    return [buf[:n0].reshape(like[0].shape).contiguous(), buf[n0:].reshape(like[1].shape).contiguous()]


def exchange_dist(rank: SlabRank, dist, group=None):
    """Halo exchange of one process per slab over torch.distributed (nccl on GPUs over NVLink, gloo in the CPU tests):
    point-to-point only, one packed [Ex plane | Ey plane] message per neighbour and direction, posted as a batch so that
    the two directions overlap.  torch.distributed rank == slab rank."""
    m = rank.meta
    ops, recv = [], {}
    if m.has_above:
        up = rank.planes_up()
        send_up = _pack(up)
        recv["hi"] = (send_up.new_empty(send_up.shape), up)
        ops += [dist.P2POp(dist.isend, send_up, m.rank + 1, group), dist.P2POp(dist.irecv, recv["hi"][0], m.rank + 1, group)]
    if m.has_below:
        down = rank.planes_down()
        send_down = _pack(down)
        recv["lo"] = (send_down.new_empty(send_down.shape), down)
        ops += [dist.P2POp(dist.isend, send_down, m.rank - 1, group), dist.P2POp(dist.irecv, recv["lo"][0], m.rank - 1, group)]
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    if "lo" in recv:
        rank.set_wall_lo(_unpack(*recv["lo"]))
    if "hi" in recv:
        rank.set_wall_hi(_unpack(*recv["hi"]))


def make_ranks_inprocess(p, n_ranks: int, **em_kw) -> List[SlabRank]:
    """all slab contexts of p in this process, on one GPU (tests; a real run has one process and GPU per slab)"""
    from .binding import EM
    out = []
    for r in range(n_ranks):
        s, meta = sub_problem(p, r, n_ranks)
        out.append(SlabRank(EM(s, **em_kw), meta))
    return out


def step_inprocess(ranks: Sequence[SlabRank], n: int = 1):
    for _ in range(n):
        for r in ranks:
            r.em.em_step(1)
        exchange_inprocess(ranks)


def gather_inprocess(ranks: Sequence[SlabRank]):
    """(six global field arrays, global power map, global energy-density map) from the owned parts"""
    parts = [r.owned_fields() for r in ranks]
    fields = [np.concatenate([pt[c] for pt in parts], axis=0) for c in range(6)]
    jl = [r.owned_joule() for r in ranks]
    return fields, np.concatenate([j[0] for j in jl], axis=0), np.concatenate([j[1] for j in jl], axis=0)
