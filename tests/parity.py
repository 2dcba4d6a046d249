"""Helpers of the GPU-vs-oracle parity tests (metric: SURVEY.md 8(c) C16)."""
import copy

import numpy as np

TOL = {64: 1e-12, 32: 2e-5}      # BASELINE.json north_star: rel-L2 <= 1e-12 (fp64), <= 2e-5 (fp32)


def rel_l2(got, want):
    """||got - want||_2 / ||want||_2 over a list of arrays (concatenated); 0/0 -> 0."""
    num = sum(float(np.sum((np.asarray(g, np.float64) - w) ** 2)) for g, w in zip(got, want))
    den = sum(float(np.sum(np.asarray(w, np.float64) ** 2)) for w in want)
    if den == 0.0:
        return 0.0 if num == 0.0 else float("inf")
    return (num / den) ** 0.5


def max_norm_err(got, want):
    """max |got - want| over a list of arrays / max |want| over the same list (the group's max-norm); 0/0 -> 0.
    A single wrong edge on a tile or chunk seam is invisible in a whole-field rel-L2 but not here."""
    num = den = 0.0
    for g, w in zip(got, want):
        w = np.asarray(w, np.float64)
        step = max(1, (1 << 24) // max(1, int(np.prod(w.shape[1:]))))       # slabs of <= 16 M values
        for k in range(0, w.shape[0], step):
            num = max(num, float(np.max(np.abs(np.asarray(g[k:k + step], np.float64) - w[k:k + step]), initial=0.0)))
            den = max(den, float(np.max(np.abs(w[k:k + step]), initial=0.0)))
    if den == 0.0:
        return 0.0 if num == 0.0 else float("inf")
    return num / den


def compare_state(gpu, orc, tol, check_zero_groups=True):
    """gpu: paper_2603_07038_b200.EM, orc: oracle.emo.Oracle, both after the same number of steps.
    Returns dict of the parity numbers (rel-L2 per group and the max-abs-diff / max-norm beside each) and asserts them."""
    Fg, Fo = gpu.fields(), orc.fields()
    eE = rel_l2(Fg[:3], Fo[:3]); eH = rel_l2(Fg[3:], Fo[3:])
    mE = max_norm_err(Fg[:3], Fo[:3]); mH = max_norm_err(Fg[3:], Fo[3:])
    pg, qg, Qg = gpu.joule_maps()
    po, qo, Qo = orc.joule()
    eq = rel_l2([qg], [qo]); ep = rel_l2([pg], [po])
    mq = max_norm_err([qg], [qo])
    eQ = abs(Qg - Qo) / abs(Qo) if Qo != 0 else abs(Qg)
    res = dict(E=eE, H=eH, q=eq, p=ep, Q=eQ, Emax=mE, Hmax=mH, qmax=mq)
    assert eE <= tol and eH <= tol, res
    assert eq <= tol and eQ <= tol and ep <= 2 * tol, res
    assert mE <= tol and mH <= tol and mq <= tol, res     # max |diff| / max |field|: a wrong seam edge shows here
    if check_zero_groups:      # components identically zero in the oracle stay (relatively) zero
        for grp in (range(0, 3), range(3, 6)):
            mx = max(float(np.max(np.abs(Fo[c]))) for c in grp)
            for c in grp:
                if not np.any(Fo[c]):
                    assert float(np.max(np.abs(Fg[c]))) <= tol * mx, (c, res)
    return res


def subbox_problem(p, lo, hi, fields):
    """Problem restricted to cells [lo, hi) (i, j, k order) with `fields` (six dense arrays of the
    box's logical shapes) as the initial state and the ports whose edges lie inside the box."""
    (i0, j0, k0), (i1, j1, k1) = lo, hi
    b = copy.copy(p)
    b.nx, b.ny, b.nz = i1 - i0, j1 - j0, k1 - k0
    b.dx, b.dy, b.dz = p.dx[i0:i1].copy(), p.dy[j0:j1].copy(), p.dz[k0:k1].copy()
    b.mat_id = np.ascontiguousarray(p.mat_id[k0:k1, j0:j1, i0:i1])
    b.init = {c: np.ascontiguousarray(f, np.float64) for c, f in enumerate(fields)}
    ext = [(b.nx, b.ny + 1, b.nz + 1), (b.nx + 1, b.ny, b.nz + 1), (b.nx + 1, b.ny + 1, b.nz)]
    eb, ee, amp, wo, wl, comp, ijk, wt = [], [], [], [], [], [], [], []
    for q in range(p.n_ports):
        start = len(comp)
        for e in range(int(p.port_edge_begin[q]), int(p.port_edge_end[q])):
            c = int(p.edge_comp[e]); i, j, k = (int(v) for v in p.edge_ijk[e])
            li, lj, lk = i - i0, j - j0, k - k0
            sx, sy, sz = ext[c]
            # strictly inside the box in the two transverse directions (box walls are PEC)
            inside = 0 <= li < sx and 0 <= lj < sy and 0 <= lk < sz
            if inside:
                if c != 0 and (li == 0 or li == b.nx): inside = False
                if c != 1 and (lj == 0 or lj == b.ny): inside = False
                if c != 2 and (lk == 0 or lk == b.nz): inside = False
            if inside:
                comp.append(c); ijk.append((li, lj, lk)); wt.append(float(p.edge_weight[e]))
        if len(comp) > start:
            eb.append(start); ee.append(len(comp)); amp.append(float(p.port_amplitude[q]))
            wo.append(int(p.port_wave_offset[q])); wl.append(int(p.port_wave_len[q]))
    b.port_edge_begin = np.asarray(eb, np.int64); b.port_edge_end = np.asarray(ee, np.int64)
    b.port_amplitude = np.asarray(amp, np.float64)
    b.port_wave_offset = np.asarray(wo, np.int64); b.port_wave_len = np.asarray(wl, np.int64)
    b.edge_comp = np.asarray(comp, np.int32); b.edge_ijk = np.asarray(ijk, np.int32).reshape(-1, 3)
    b.edge_weight = np.asarray(wt, np.float64)
    return b
