"""Test-side discrete calculus on the staggered grid, written independently of oracle/ and of
the CUDA path (vectorised NumPy / SciPy sparse incidence matrices).  Used by the pins to
evaluate invariants (energy, Poynting balance, divergences) and to assemble the paper's
eq. (1)-(3) operators literally for the dense brute force.
"""
import numpy as np
import scipy.sparse as sp


def shapes(nx, ny, nz):
    return [(nz + 1, ny + 1, nx), (nz + 1, ny, nx + 1), (nz, ny + 1, nx + 1),
            (nz, ny, nx + 1), (nz, ny + 1, nx), (nz + 1, ny, nx)]


def dual(d):
    """dual (centre-to-centre) lengths, half cells at both ends; length n+1"""
    d = np.asarray(d, np.float64)
    t = np.empty(d.shape[0] + 1)
    t[0] = 0.5 * d[0]; t[-1] = 0.5 * d[-1]
    t[1:-1] = 0.5 * (d[:-1] + d[1:])
    return t


def _pad(a, axes):
    pw = [(1, 1) if ax in axes else (0, 0) for ax in range(3)]
    return np.pad(a, pw)


def edge_mean(cell, dx, dy, dz, comp):
    """area-weighted mean of a cell quantity over the <=4 cells round each edge of direction comp
    (SURVEY.md 8(c) C5).  cell: (nz, ny, nx).  Returns the array in the edge's logical shape."""
    nz, ny, nx = cell.shape
    wx = np.pad(dx, 1); wy = np.pad(dy, 1); wz = np.pad(dz, 1)
    if comp == 0:      # Ex: average over (j-1, j) x (k-1, k)
        c = _pad(cell, (0, 1)); num = 0; den = 0
        for b in (0, 1):
            for a in (0, 1):
                w = wz[b:b + nz + 1][:, None, None] * wy[a:a + ny + 1][None, :, None]
                num = num + w * c[b:b + nz + 1, a:a + ny + 1, :]; den = den + w
        return num / (den + 0 * num)
    if comp == 1:      # Ey: (i-1, i) x (k-1, k)
        c = _pad(cell, (0, 2)); num = 0; den = 0
        for b in (0, 1):
            for a in (0, 1):
                w = wz[b:b + nz + 1][:, None, None] * wx[a:a + nx + 1][None, None, :]
                num = num + w * c[b:b + nz + 1, :, a:a + nx + 1]; den = den + w
        return num / (den + 0 * num)
    c = _pad(cell, (1, 2)); num = 0; den = 0
    for b in (0, 1):
        for a in (0, 1):
            w = wy[b:b + ny + 1][None, :, None] * wx[a:a + nx + 1][None, None, :]
            num = num + w * c[:, b:b + ny + 1, a:a + nx + 1]; den = den + w
    return num / (den + 0 * num)


def face_mean(cell, dx, dy, dz, comp):
    """length-weighted mean over the <=2 cells across each face normal to comp."""
    nz, ny, nx = cell.shape
    if comp == 0:
        w = np.pad(dx, 1); c = _pad(cell, (2,))
        num = sum(w[a:a + nx + 1][None, None, :] * c[:, :, a:a + nx + 1] for a in (0, 1))
        den = sum(w[a:a + nx + 1] for a in (0, 1))[None, None, :]
    elif comp == 1:
        w = np.pad(dy, 1); c = _pad(cell, (1,))
        num = sum(w[a:a + ny + 1][None, :, None] * c[:, a:a + ny + 1, :] for a in (0, 1))
        den = sum(w[a:a + ny + 1] for a in (0, 1))[None, :, None]
    else:
        w = np.pad(dz, 1); c = _pad(cell, (0,))
        num = sum(w[a:a + nz + 1][:, None, None] * c[a:a + nz + 1, :, :] for a in (0, 1))
        den = sum(w[a:a + nz + 1] for a in (0, 1))[:, None, None]
    return num / den


def fixed_mask(nx, ny, nz, comp, pec_cell=None, bc=(0,) * 6):
    """True on PEC-fixed edges (tangential E on the walls whose bc is PEC = 0, or touching a PEC-flagged
    cell).  bc order: -x, +x, -y, +y, -z, +z; 1 = PMC (the wall's tangential E stays an unknown)."""
    sh = shapes(nx, ny, nz)[comp]
    m = np.zeros(sh, bool)
    x0, x1, y0, y1, z0, z1 = (b == 0 for b in bc)
    if comp == 0:
        m[0, :, :] |= z0; m[-1, :, :] |= z1; m[:, 0, :] |= y0; m[:, -1, :] |= y1
    elif comp == 1:
        m[0, :, :] |= z0; m[-1, :, :] |= z1; m[:, :, 0] |= x0; m[:, :, -1] |= x1
    else:
        m[:, 0, :] |= y0; m[:, -1, :] |= y1; m[:, :, 0] |= x0; m[:, :, -1] |= x1
    if pec_cell is not None and pec_cell.any():
        one = np.ones(1)
        touched = edge_mean(pec_cell.astype(np.float64), np.ones(nx), np.ones(ny), np.ones(nz), comp)
        m |= np.nan_to_num(touched) > 0
    return m


class Geometry:
    """edge lengths, dual-face areas, face areas, dual-edge lengths for all six components"""

    def __init__(self, dx, dy, dz):
        dx = np.asarray(dx, np.float64); dy = np.asarray(dy, np.float64); dz = np.asarray(dz, np.float64)
        tx, ty, tz = dual(dx), dual(dy), dual(dz)
        X = lambda v: v[None, None, :]; Y = lambda v: v[None, :, None]; Z = lambda v: v[:, None, None]
        self.len_e = [X(dx) + 0 * Y(ty) + 0 * Z(tz), Y(dy) + 0 * X(tx) + 0 * Z(tz), Z(dz) + 0 * X(tx) + 0 * Y(ty)]
        self.area_dual = [Y(ty) * Z(tz) + 0 * X(dx), X(tx) * Z(tz) + 0 * Y(dy), X(tx) * Y(ty) + 0 * Z(dz)]
        self.area_f = [Y(dy) * Z(dz) + 0 * X(tx), X(dx) * Z(dz) + 0 * Y(ty), X(dx) * Y(dy) + 0 * Z(tz)]
        self.len_dual = [X(tx) + 0 * Y(dy) + 0 * Z(dz), Y(ty) + 0 * X(dx) + 0 * Z(dz), Z(tz) + 0 * X(dx) + 0 * Y(dy)]
        self.vol = Z(dz) * Y(dy) * X(dx)


def energy(E, Hm, Hp, eps_e, nu_f, geo):
    """Conserved discrete energy:
    1/2 sum_e eps_e E_e^2 l_e A~_e + 1/2 sum_f (1/nu_f) H_f^{n+1/2} H_f^{n-1/2} A_f l~_f"""
    tot = 0.0
    for a in range(3):
        tot += 0.5 * np.sum(np.nan_to_num(eps_e[a]) * E[a] ** 2 * geo.len_e[a] * geo.area_dual[a])
        tot += 0.5 * np.sum(Hm[a] * Hp[a] / nu_f[a] * geo.area_f[a] * geo.len_dual[a])
    return tot


# ---- incidence-based curl matrices (edges/faces numbered in logical array order, Ex|Ey|Ez) ----
class Operators:
    def __init__(self, nx, ny, nz, dx, dy, dz):
        self.n = (nx, ny, nz)
        sh = shapes(nx, ny, nz)
        self.sh = sh
        ne = [int(np.prod(s)) for s in sh[:3]]; nf = [int(np.prod(s)) for s in sh[3:]]
        self.eoff = np.concatenate([[0], np.cumsum(ne)]); self.foff = np.concatenate([[0], np.cumsum(nf)])
        tx, ty, tz = dual(dx), dual(dy), dual(dz)
        d = [np.asarray(dx, float), np.asarray(dy, float), np.asarray(dz, float)]
        t = [tx, ty, tz]

        def eidx(c, i, j, k):
            s = sh[c]; return self.eoff[c] + (k * s[1] + j) * s[2] + i

        def fidx(c, i, j, k):
            s = sh[3 + c]; return self.foff[c] + (k * s[1] + j) * s[2] + i
        self.eidx, self.fidx = eidx, fidx
        # C_e: for each face, circulation of E round its boundary (right-handed about +normal) / area
        rows, cols, vals = [], [], []
        for c in range(3):
            a, b = (c + 1) % 3, (c + 2) % 3          # face normal c spans directions a, b
            s = sh[3 + c]
            for k in range(s[0]):
                for j in range(s[1]):
                    for i in range(s[2]):
                        p = [i, j, k]
                        f = fidx(c, i, j, k)
                        la, lb = d[a][p[a]], d[b][p[b]]
                        area = la * lb
                        # (curl E)_c = dE_b/da - dE_a/db
                        pa = list(p); pa[a] += 1
                        pb = list(p); pb[b] += 1
                        for (comp, q, sign, ln) in ((b, pa, +1, lb), (b, p, -1, lb), (a, pb, -1, la), (a, p, +1, la)):
                            rows.append(f); cols.append(eidx(comp, *q)); vals.append(sign * ln / area)
        self.Ce = sp.csr_matrix((vals, (rows, cols)), shape=(self.foff[-1], self.eoff[-1]))
        # C_h: for each edge, circulation of H round the dual face / dual area; H outside the
        # domain does not exist (such rows belong to PEC-fixed edges and are removed later)
        rows, cols, vals = [], [], []
        for c in range(3):
            a, b = (c + 1) % 3, (c + 2) % 3
            s = sh[c]
            for k in range(s[0]):
                for j in range(s[1]):
                    for i in range(s[2]):
                        p = [i, j, k]
                        e = eidx(c, i, j, k)
                        ta, tb = t[a][p[a]], t[b][p[b]]
                        area = ta * tb
                        pa = list(p); pa[a] -= 1
                        pb = list(p); pb[b] -= 1
                        # (curl H)_c = dH_b/da - dH_a/db with backward differences
                        for (comp, q, sign, ln) in ((b, p, +1, tb), (b, pa, -1, tb), (a, p, -1, ta), (a, pb, +1, ta)):
                            sf = sh[3 + comp]
                            if min(q) < 0 or q[0] >= sf[2] or q[1] >= sf[1] or q[2] >= sf[0]:
                                continue
                            rows.append(e); cols.append(fidx(comp, *q)); vals.append(sign * ln / area)
        self.Ch = sp.csr_matrix((vals, (rows, cols)), shape=(self.eoff[-1], self.foff[-1]))

    def flat(self, arrs):
        return np.concatenate([np.asarray(a, np.float64).ravel() for a in arrs])

    def unflat_e(self, v):
        return [v[self.eoff[c]:self.eoff[c + 1]].reshape(self.sh[c]) for c in range(3)]
