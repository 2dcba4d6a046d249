"""P7: dense-matrix brute force of the paper's eq. (1)-(3) on a 4x4x4 mesh (north_star check 5).

The second-order E-only recurrence  M e^{n+1} = N e^n - K e^{n-1} - dt^2 (dJ/dt)^n  with
M = D_eps + dt/2 D_sigma, N = 2 D_eps - dt^2 S, K = D_eps - dt/2 D_sigma, S = C_h D_nu C_e
 is iterated literally with dense matrices assembled from the incidence
definition (tests/discrete.py), starting from e^0 = e^{-1} = 0, and compared with the leapfrog
oracle.  This pins readings C2 (E/H leapfrog == eq. 2), C3 (dJ/dt as a centred half-step
difference), C4 (start-up), C5 (material averaging) and C6 (CD loss) of SURVEY.md 8(c) at once.
"""
import numpy as np
import pytest

import workloads as W
from workloads.problem import LOSS_CD
from oracle import emo
import discrete as D


@pytest.mark.parametrize("dims,seed,bc", [((4, 4, 4), 101, (0,) * 6), ((3, 5, 4), 102, (0,) * 6),
                                          ((4, 4, 4), 104, (1, 0, 0, 1, 1, 0)), ((3, 4, 5), 105, (1,) * 6)])
def test_p7_dense_eq2_eq3(dims, seed, bc):
    """bc with 1 = PMC walls: their tangential edges stay in the free set; C_h built from
    the incidence definition already has the half dual faces and no H outside the domain."""
    nx, ny, nz = dims
    steps = 300
    p = W.random_problem(nx, ny, nz, seed=seed, loss_mode=LOSS_CD, steps=steps, n_ports=2, blocky=False, bc=bc)
    p.init = None                                              # e^0 = e^{-1} = 0, H^{-1/2} = 0
    assert p.n_ports >= 1
    ops = D.Operators(nx, ny, nz, p.dx, p.dy, p.dz)
    eps_e = ops.flat([D.edge_mean(p.table[p.mat_id, 0], p.dx, p.dy, p.dz, a) for a in range(3)])
    sig_e = ops.flat([D.edge_mean(p.table[p.mat_id, 2], p.dx, p.dy, p.dz, a) for a in range(3)])
    nu_f = ops.flat([D.face_mean(1.0 / p.table[p.mat_id, 1], p.dx, p.dy, p.dz, a) for a in range(3)])
    free = ~ops.flat([D.fixed_mask(nx, ny, nz, a, bc=p.bc) for a in range(3)]).astype(bool)
    Ce = ops.Ce.toarray(); Ch = ops.Ch.toarray()
    if dims == (4, 4, 4):
        assert Ce.shape == (240, 300) and Ch.shape == (300, 240)
    S = (Ch @ np.diag(nu_f) @ Ce)[np.ix_(free, free)]
    dt = p.dt
    De, Ds = np.diag(eps_e[free]), np.diag(sig_e[free])
    M = De + 0.5 * dt * Ds
    N = 2 * De - dt * dt * S
    K = De - 0.5 * dt * Ds
    Minv = np.diag(1.0 / np.diag(M))

    def J_half(n):          # J^{n+1/2} on all edges, 0 for n < 0
        J = np.zeros(ops.eoff[-1])
        if n < 0:
            return J
        for pt in range(p.n_ports):
            w = p.wave[p.port_wave_offset[pt] + n] if n < p.port_wave_len[pt] else 0.0
            for e in range(p.port_edge_begin[pt], p.port_edge_end[pt]):
                c = int(p.edge_comp[e]); i, j, k = (int(v) for v in p.edge_ijk[e])
                J[ops.eidx(c, i, j, k)] += p.port_amplitude[pt] * p.edge_weight[e] * w
        return J

    e_prev = np.zeros(int(free.sum())); e_cur = np.zeros_like(e_prev)
    for n in range(steps):
        dJ = (J_half(n) - J_half(n - 1))[free] / dt
        e_next = Minv @ (N @ e_cur - K @ e_prev - dt * dt * dJ)
        e_prev, e_cur = e_cur, e_next
    o = emo.Oracle(p)
    o.step(steps)
    got = ops.flat(o.fields()[:3])
    assert np.all(got[~free] == 0.0)
    err = np.linalg.norm(got[free] - e_cur) / np.linalg.norm(e_cur)
    assert np.linalg.norm(e_cur) > 0
    assert err < 5e-12, err


def test_weighted_curlcurl_is_symmetric_psd():
    """C5 consequence: W_e S (W_e = edge length x dual area) is symmetric positive semi-definite,
    i.e. C_h = W_e^-1 C_e^T W_f -- the adjointness that makes P2 hold on non-uniform grids."""
    nx, ny, nz = 4, 3, 5
    p = W.random_problem(nx, ny, nz, seed=103, n_ports=0)
    ops = D.Operators(nx, ny, nz, p.dx, p.dy, p.dz)
    geo = D.Geometry(p.dx, p.dy, p.dz)
    We = ops.flat([geo.len_e[a] * geo.area_dual[a] for a in range(3)])
    nu_f = ops.flat([D.face_mean(1.0 / p.table[p.mat_id, 1], p.dx, p.dy, p.dz, a) for a in range(3)])
    free = ~ops.flat([D.fixed_mask(nx, ny, nz, a) for a in range(3)]).astype(bool)
    S = (ops.Ch.toarray() @ np.diag(nu_f) @ ops.Ce.toarray())
    A = (np.diag(We) @ S)[np.ix_(free, free)]
    assert np.max(np.abs(A - A.T)) < 1e-12 * np.max(np.abs(A))
    assert np.linalg.eigvalsh(0.5 * (A + A.T)).min() > -1e-10 * np.max(np.abs(A))
