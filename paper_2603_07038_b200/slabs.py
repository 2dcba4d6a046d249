"""z-slab decomposition of the EM time-marching over several GPUs (NEXT-3 of SURVEY.md 8(f)).

One process per GPU, each with its own em_ctx over its slab of cell layers [a, b) EXTENDED by one ghost cell layer on
every interior side.  The artificial end walls of the extended slab are PMC walls (include/em.h EM_BC_PMC): their
tangential E (Ex, Ey on the wall's node plane) is an unknown that the library lets the caller overwrite, and it is
the ONLY field value a slab cannot compute itself -- everything one plane inside the wall (H', E'z of the ghost layer,
the Joule sum that closes on the plane above) follows from correct inputs.  So the halo after every step is
    to the slab above : my Ex, Ey at global node plane b-1   -> its lower wall plane
    to the slab below : my Ex, Ey at global node plane a+1   -> its upper wall plane
(2 x nx*ny reals per neighbour), point-to-point only; with the two-way thermal coupling the temperature
rise of the owned boundary layer rides along (-> the neighbour's ghost layer, whose theta and sigma(T) feed the owned
layer's conduction and edge conductivities); with theta on the mesh NODES (the paper's placement) it is the temperature
rise of the same node plane as Ex, Ey that rides along (-> the neighbour's wall plane, the only nodes it cannot update).  Two ways to move it, both with every arithmetic step in the CUDA kernels:

  mode "p2p"  : em_get_halo packs the message with one kernel into a preallocated buffer, torch.distributed moves it
                (batched isend/irecv: NCCL over NVLink, stream-ordered, no host synchronisation; gloo in the CPU tests),
                em_set_halo unpacks with one kernel.  Works for the coupled step too.
  mode "peer" : the halo is FUSED into the sweep: the kernel stores E'x, E'y of the plane the neighbour needs straight
                into the neighbour's wall plane through a peer mapping of its workspace (em_set_peer_halo; NVLink
                stores, CUDA IPC between processes), overlapped with the sweep by construction; the only thing left
                per step is one tiny stream-ordered all-reduce as the cross-rank barrier (step n+1 of a rank may start
                only when its neighbours finished step n).

The Joule total is the all-reduced sum of the owned layers' totals (em_joule_layers).  The path of BASELINE.json is one
GPU; this is the scale-out of the same kernels, tested on one GPU (slab contexts run one after another; two processes
sharing one GPU for the IPC wiring) and, for the exchange logic, with gloo on CPU.
"""
from __future__ import annotations

import copy
import dataclasses
from typing import List, Optional, Sequence

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


def slab_meta(nz: int, rank: int, n_ranks: int) -> SlabMeta:
    a, b = slab_ranges(nz, n_ranks)[rank]
    return SlabMeta(rank, n_ranks, a, b, a - 1 if rank > 0 else 0, b + 1 if rank < n_ranks - 1 else nz, nz)


def sub_problem(p, rank: int, n_ranks: int):
    """The inputs of slab `rank`: a shallow copy of the problem restricted to the extended slab, with PMC on the
    artificial walls, the port edges that fall inside it (k shifted) and the matching slices of the initial fields."""
    meta = slab_meta(p.nz, rank, n_ranks)
    lo, hi = meta.lo, meta.hi
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
    """One slab: its context (paper_2603_07038_b200.EM, or anything with em_step / em_get_halo / em_set_halo /
    new_halo_buffer) and the plane bookkeeping of the halo."""

    def __init__(self, em, meta: SlabMeta, mode: str = "p2p"):
        assert mode in ("p2p", "peer")
        self.em, self.meta, self.mode = em, meta, mode
        self._buf = {}
        self._token = None
        # False until the wall planes hold the neighbours' values of the CURRENT state.  A slab cannot apply the whole-domain
        # rules to its wall plane by itself: an initial Ex, Ey there that the single-domain em_set_field would force to 0
        # because the edge touches a PEC-flagged cell ABOVE the plane -- a cell this slab does not hold -- stays as given.
        # The neighbour holds that plane as an interior one, correctly masked, so one exchange before the first step
        # settles it (found by the random slab campaign of tests/test_emu_sweep.py).  Set it to False again after
        # em_set_field / em_set_temperature_rise on a slab context.
        self.halo_synced = False

    # local indices --------------------------------------------------------------------------------------------
    @property
    def nz_local(self) -> int:
        return self.meta.hi - self.meta.lo

    @property
    def k_send_up(self) -> int:        # global node plane b - 1
        return self.meta.b - 1 - self.meta.lo

    @property
    def k_send_down(self) -> int:      # global node plane a + 1
        return self.meta.a + 1 - self.meta.lo

    @property
    def layer_send_up(self) -> int:    # my top owned cell layer b - 1 -> the ghost layer of the slab above
        return self.meta.b - 1 - self.meta.lo

    @property
    def layer_send_down(self) -> int:  # my bottom owned cell layer a -> the ghost layer of the slab below
        return self.meta.a - self.meta.lo

    @property
    def k_wall_lo(self) -> int:
        return 0

    @property
    def k_wall_hi(self) -> int:
        return self.nz_local

    def buf(self, name):
        if name not in self._buf:
            self._buf[name] = self.em.new_halo_buffer()
        return self._buf[name]

    # the halo in two kernels per neighbour ---------------------------------------------------------------------------
    def pack_up(self):
        return self.em.em_get_halo(self.k_send_up, self.layer_send_up, self.buf("send_up"))

    def pack_down(self):
        return self.em.em_get_halo(self.k_send_down, self.layer_send_down, self.buf("send_down"))

    def unpack_lo(self, msg):          # from the slab below: my lower wall plane and my ghost layer 0
        self.em.em_set_halo(self.k_wall_lo, 0, msg)

    def unpack_hi(self, msg):          # from the slab above: my upper wall plane and my ghost layer nz_local - 1
        self.em.em_set_halo(self.k_wall_hi, self.nz_local - 1, msg)

    # stepping with torch.distributed (rank == slab rank) ---------------------------------------------------------
    def step(self, n: int, dist, group=None):
        if not self.halo_synced:
            exchange_dist(self, dist, group)              # (pack / unpack kernels, whatever the transport of the steps)
            self.halo_synced = True
            if self.mode == "peer":
                barrier_on_stream(self, dist, group)      # the neighbours' sweeps store into my planes from step 1 on
        for _ in range(n):
            self.em.em_step(1)
            if self.mode == "p2p":
                exchange_dist(self, dist, group)
            else:
                barrier_on_stream(self, dist, group)

    def reset(self):
        self.em.em_reset()

    def joule_total(self, dist=None, group=None) -> float:
        """Joule energy of the WHOLE problem: the owned layers' total, all-reduced over the ranks."""
        own = self.em.em_joule_layers(self.meta.a - self.meta.lo, self.meta.b - self.meta.lo)
        if dist is None:
            return own
        import torch
        t = torch.tensor([own], dtype=torch.float64, device=self.em.device if dist.get_backend(group) == "nccl" else "cpu")
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
        return float(t.item())

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

    def owned_theta(self):
        """per-cell stage: the owned cell layers; nodal stage: node planes a .. b-1 (the last slab also owns plane nz)"""
        m = self.meta
        th = self.em.em_get_temperature_rise()
        nodal = th.shape[0] == self.nz_local + 1
        return th[m.a - m.lo:m.b - m.lo + (1 if nodal and not m.has_above else 0)]


def exchange_dist(rank: SlabRank, dist, group=None):
    """Halo exchange of one process per slab over torch.distributed (nccl on GPUs over NVLink, gloo in the CPU tests):
    point-to-point only, one packed message per neighbour and direction in preallocated buffers, posted as one batch so
    that the two directions overlap.  With nccl everything is stream-ordered (wait() makes the current stream wait)."""
    m = rank.meta
    ops = []
    # (a backend without device-to-device send / recv -- gloo with CUDA buffers, i.e. the one-GPU IPC test -- goes through
    # host copies of the packed messages; nccl and the CPU tests move the buffers themselves)
    staged = []
    def out(t):
        return t if (t.device.type == "cpu" or dist.get_backend(group) == "nccl") else t.cpu()
    def into(t):
        if t.device.type == "cpu" or dist.get_backend(group) == "nccl":
            return t
        staged.append((t, t.cpu()))
        return staged[-1][1]
    if m.has_above:
        ops += [dist.P2POp(dist.isend, out(rank.pack_up()), m.rank + 1, group),
                dist.P2POp(dist.irecv, into(rank.buf("recv_hi")), m.rank + 1, group)]
    if m.has_below:
        ops += [dist.P2POp(dist.isend, out(rank.pack_down()), m.rank - 1, group),
                dist.P2POp(dist.irecv, into(rank.buf("recv_lo")), m.rank - 1, group)]
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    for dev, host in staged:
        dev.copy_(host)
    if m.has_below:
        rank.unpack_lo(rank.buf("recv_lo"))
    if m.has_above:
        rank.unpack_hi(rank.buf("recv_hi"))


def barrier_on_stream(rank: SlabRank, dist, group=None):
    """The cross-rank barrier of the peer mode: nccl -- a one-element all-reduce, stream-ordered, no host
    synchronisation; any other backend -- device synchronise, then a host barrier."""
    import torch
    if dist.get_backend(group) == "nccl":
        if rank._token is None:
            rank._token = torch.zeros(1, dtype=torch.float32, device=rank.em.device)
        dist.all_reduce(rank._token, group=group)
    else:
        torch.cuda.synchronize(rank.em.device)
        dist.barrier(group)


# ---- peer wiring ------------------------------------------------------------------------------------------------------
def _peer_addresses(base_ptr: int, offsets):
    return [base_ptr + int(o) for o in offsets]


def connect_peers_inprocess(ranks: Sequence[SlabRank]):
    """All slab contexts live in this process on one GPU: a neighbour's workspace is directly addressable."""
    for n, r in enumerate(ranks):
        if r.meta.has_above:
            nb = ranks[n + 1]
            r.em.em_set_peer_halo(1, r.k_send_up, _peer_addresses(nb.em.workspace_ptr, nb.em.wall_offsets(0)))
        if r.meta.has_below:
            nb = ranks[n - 1]
            r.em.em_set_peer_halo(0, r.k_send_down, _peer_addresses(nb.em.workspace_ptr, nb.em.wall_offsets(1)))
        r.mode = "peer"


def connect_peers_dist(rank: SlabRank, dist, group=None):
    """One process per slab: every rank exports its workspace as a CUDA IPC handle (torch's storage sharing), the
    neighbours map it (NVLink peer mapping between GPUs of one node) and hand the wall-plane addresses to their sweeps."""
    import torch
    em = rank.em
    storage = em._ws.untyped_storage()
    info = {"ipc": storage._share_cuda_(), "ws_off": em.workspace_ptr - storage.data_ptr(),
            "wall_lo": em.wall_offsets(0), "wall_hi": em.wall_offsets(1)}
    world = dist.get_world_size(group)
    infos: List[Optional[dict]] = [None] * world
    dist.all_gather_object(infos, info, group=group)
    rank._peer_storages = []                                # keep the mappings alive
    m = rank.meta
    for side, nb in ((1, m.rank + 1 if m.has_above else None), (0, m.rank - 1 if m.has_below else None)):
        if nb is None:
            continue
        st = torch.UntypedStorage._new_shared_cuda(*infos[nb]["ipc"])
        rank._peer_storages.append(st)
        base = st.data_ptr() + infos[nb]["ws_off"]
        offs = infos[nb]["wall_lo"] if side == 1 else infos[nb]["wall_hi"]       # my +z neighbour's -z wall and vice versa
        em.em_set_peer_halo(side, rank.k_send_up if side == 1 else rank.k_send_down, _peer_addresses(base, offs))
    rank.mode = "peer"
    torch.cuda.synchronize(em.device)
    dist.barrier(group)


# ---- all slabs in one process on one GPU (tests) -----------------------------------------------------------------------
def exchange_inprocess(ranks: Sequence[SlabRank]):
    """Halo exchange between slab contexts that live in ONE process (one GPU, run one after another): the packed
    messages are handed over directly (pack kernel -> unpack kernel)."""
    ups = [r.pack_up() if r.meta.has_above else None for r in ranks]
    downs = [r.pack_down() if r.meta.has_below else None for r in ranks]
    for n, r in enumerate(ranks):
        if r.meta.has_below:
            r.unpack_lo(ups[n - 1])
        if r.meta.has_above:
            r.unpack_hi(downs[n + 1])


def make_ranks_inprocess(p, n_ranks: int, mode: str = "p2p", **em_kw) -> List[SlabRank]:
    """all slab contexts of p in this process, on one GPU (tests; a real run has one process and GPU per slab)"""
    from .binding import EM
    out = []
    for r in range(n_ranks):
        s, meta = sub_problem(p, r, n_ranks)
        out.append(SlabRank(EM(s, **em_kw), meta))
    if mode == "peer":
        connect_peers_inprocess(out)
    return out


def step_inprocess(ranks: Sequence[SlabRank], n: int = 1):
    if not all(r.halo_synced for r in ranks):
        exchange_inprocess(ranks)                   # wall planes of the initial state (SlabRank.halo_synced)
        for r in ranks:
            r.halo_synced = True
    for _ in range(n):
        for r in ranks:
            r.em.em_step(1)
        if ranks[0].mode == "p2p":
            exchange_inprocess(ranks)           # (peer mode: the sweeps stored the halos themselves; one stream orders them)


def gather_inprocess(ranks: Sequence[SlabRank]):
    """(six global field arrays, global power map, global energy-density map) from the owned parts"""
    parts = [r.owned_fields() for r in ranks]
    fields = [np.concatenate([pt[c] for pt in parts], axis=0) for c in range(6)]
    jl = [r.owned_joule() for r in ranks]
    return fields, np.concatenate([j[0] for j in jl], axis=0), np.concatenate([j[1] for j in jl], axis=0)
