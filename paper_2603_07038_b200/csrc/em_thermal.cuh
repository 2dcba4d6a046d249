// em_thermal.cuh -- two-way EM-thermal coupling (NEXT-1 of SURVEY.md 8(f); eq. (4)-(6), L84-L96) on the
// split kernel strategy: a first correct CUDA path, not yet fused into the sweep.
//
//   eq. (5)  theta' = theta - dt/(rho c_p) (M_kk theta) + dq/(rho c_p)        theta = T - T0 per cell
//   eq. (6)  sigma' = sigma_0 / (1 + alpha theta')                            feeds D_sigma of the next E update (L78)
//
// dq = the Joule energy density deposited in this step (a4, time-centred, with the sigma(T^n) the E update used);
// M_kk = V0a^T D_k V0 as the cell-centred finite-volume -div k grad with the series conductivity of the two half
// cells on every face and no flux through the walls (readings T1-T5).  The per-cell conductivity lives in
// an array of the common padded geometry (0 in the pad), so the E update gathers it exactly like the table's sigma.
#pragma once
#include "em_split.cuh"
#include <type_traits>

namespace em {

// (ThEntry: em_common.cuh)

template <typename R>
struct ThermalParams {
    R *theta, *theta_n;          // temperature rise, ping-pong
    R *sig;                      // current sigma per cell
    const ThEntry<R> *ttable;    // n_table entries
};

// Edge coefficients with the per-cell sigma array instead of the table's sigma (same arithmetic as edge_coeffs).
template <typename R, int LOSS>
__device__ __forceinline__ void edge_coeffs_sig(const MatEntry<R> *tab, const uint8_t *mat, const R *sig, long long o,
                                                long long PX, long long PXY, R fx, R fy, R fz, R r[3], R sg[3], R h2[3]) {
    const MatEntry<R> c000 = tab[mat[o]], c100 = tab[mat[o - 1]], c010 = tab[mat[o - PX]];
    const MatEntry<R> c110 = tab[mat[o - PX - 1]], c001 = tab[mat[o - PXY]];
    const MatEntry<R> c101 = tab[mat[o - PXY - 1]], c011 = tab[mat[o - PXY - PX]];
    const R b000 = sig[o], b100 = sig[o - 1], b010 = sig[o - PX], b110 = sig[o - PX - 1];
    const R b001 = sig[o - PXY], b101 = sig[o - PXY - 1], b011 = sig[o - PXY - PX];
    {   // Ex: cells (i, j-1..j, k-1..k)
        const R A = lerp(lerp(c011.a, c001.a, fy), lerp(c010.a, c000.a, fy), fz);
        const R B = lerp(lerp(b011, b001, fy), lerp(b010, b000, fy), fz);
        const R m = (c011.m * c001.m) * (c010.m * c000.m);
        const R rr = loss_r<R, LOSS>(A, B);
        r[0] = m * rr; sg[0] = B; h2[0] = (LOSS == 0) ? R(2) * A * rr : R(2) - rr * B;
    }
    {   // Ey: cells (i-1..i, j, k-1..k)
        const R A = lerp(lerp(c101.a, c001.a, fx), lerp(c100.a, c000.a, fx), fz);
        const R B = lerp(lerp(b101, b001, fx), lerp(b100, b000, fx), fz);
        const R m = (c101.m * c001.m) * (c100.m * c000.m);
        const R rr = loss_r<R, LOSS>(A, B);
        r[1] = m * rr; sg[1] = B; h2[1] = (LOSS == 0) ? R(2) * A * rr : R(2) - rr * B;
    }
    {   // Ez: cells (i-1..i, j-1..j, k)
        const R A = lerp(lerp(c110.a, c010.a, fx), lerp(c100.a, c000.a, fx), fy);
        const R B = lerp(lerp(b110, b010, fx), lerp(b100, b000, fx), fy);
        const R m = (c110.m * c010.m) * (c100.m * c000.m);
        const R rr = loss_r<R, LOSS>(A, B);
        r[2] = m * rr; sg[2] = B; h2[2] = (LOSS == 0) ? R(2) * A * rr : R(2) - rr * B;
    }
}

// a2 with D_sigma(T^n) -- PAPER.md eq. (2)-(3) and L78; reads E, writes En.
template <typename R, int LOSS>
__global__ void __launch_bounds__(256) k_split_e_sig(DevParams<R> p, const R *sig) {
    __shared__ MatEntry<R> s_tab[kMaxTable];
    load_table(s_tab, p);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i > p.nx || j > p.ny) return;
    const long long PX = p.PX, PXY = p.PXY;
    const long long o = ((long long)k * p.PY + j) * PX + i;
    R r[3], sg[3], h2[3];
    edge_coeffs_sig<R, LOSS>(s_tab, p.mat, sig, o, PX, PXY, p.fx[i], p.fy[j], p.fz[k], r, sg, h2);
    const R hx = p.H[0][o], hxj = p.H[0][o - PX], hxk = p.H[0][o - PXY];
    const R hy = p.H[1][o], hyi = p.H[1][o - 1], hyk = p.H[1][o - PXY];
    const R hz = p.H[2][o], hzi = p.H[2][o - 1], hzj = p.H[2][o - PX];
    const R rtx = p.rtx[i], rty = p.rty[j], rtz = p.rtz[k];
    const R ex = p.E[0][o], ey = p.E[1][o], ez = p.E[2][o];
    const R cx = (hz - hzj) * rty - (hy - hyk) * rtz;
    const R cy = (hx - hxk) * rtz - (hz - hzi) * rtx;
    const R cz = (hy - hyi) * rtx - (hx - hxj) * rty;
    p.En[0][o] = mad(r[0], mad(-sg[0], ex, cx), ex);
    p.En[1][o] = mad(r[1], mad(-sg[1], ey, cy), ey);
    p.En[2][o] = mad(r[2], mad(-sg[2], ez, cz), ez);
    p.Hn[0][o] = mad(r[0], cx, h2[0] * ex);               // E' + E without cancellation (em_split.cuh edge_coeffs)
    p.Hn[1][o] = mad(r[1], cy, h2[1] * ey);
    p.Hn[2][o] = mad(r[2], cz, h2[2] * ez);
}

// r_e of every unique source edge with the current sigma(T^n): recomputed every step in the coupled mode.
template <typename R, int LOSS>
__global__ void k_source_coef_sig(DevParams<R> p, DevSources<R> s, const R *sig) {
    const int u = blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= s.n_unique) return;
    const long long o = s.off[u];
    const long long PX = p.PX, PXY = p.PXY;
    const long long kk = o / PXY, rem = o - kk * PXY;
    const int j = (int)(rem / PX), i = (int)(rem - (long long)j * PX), k = (int)kk;
    R r[3], sg[3], h2[3];
    edge_coeffs_sig<R, LOSS>(p.table, p.mat, sig, o, PX, PXY, p.fx[i], p.fy[j], p.fz[k], r, sg, h2);
    s.r[u] = r[s.comp[u]];
}

// a4 + eq. (5) + eq. (6): Joule heat of the step into q and into the cell's temperature rise, conduction to the six
// neighbours from theta^n (ping-pong), then sigma(T^{n+1}) of the own cell.
template <typename R>
__global__ void __launch_bounds__(256) k_joule_thermal(DevParams<R> p, ThermalParams<R> t) {
    __shared__ ThEntry<R> s_th[kMaxTable];
    {
        const int tid = threadIdx.y * blockDim.x + threadIdx.x, nth = blockDim.x * blockDim.y;
        for (int m = tid; m < p.n_table; m += nth) s_th[m] = t.ttable[m];
        __syncthreads();
    }
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= p.nx || j >= p.ny) return;
    const long long PX = p.PX, PXY = p.PXY;
    const long long o = ((long long)k * p.PY + j) * PX + i;
    const ThEntry<R> me = s_th[p.mat[o]];
    const R sig = t.sig[o];
    R dq = R(0);
    if (sig != R(0)) {
        R s = 0;
#define EM_ACC(c, off) { const R t_ = p.Hn[c][o + (off)]; s = mad(t_, t_, s); }      /* E' + E as k_split_e_sig formed it */
        EM_ACC(0, 0) EM_ACC(0, PX) EM_ACC(0, PXY) EM_ACC(0, PXY + PX)
        EM_ACC(1, 0) EM_ACC(1, 1)  EM_ACC(1, PXY) EM_ACC(1, PXY + 1)
        EM_ACC(2, 0) EM_ACC(2, 1)  EM_ACC(2, PX)  EM_ACC(2, PX + 1)
#undef EM_ACC
        dq = p.dt * sig * R(0.0625) * s;
        p.q[o] += dq;
    }
    const R th = t.theta[o];
    const R rdx = p.rdx[i], rdy = p.rdy[j], rdz = p.rdz[k];
    const R gx = rdx * me.k, gy = rdy * me.k, gz = rdz * me.k;     // own half-cell conductances k/d
    R lap = R(0);                                        // (M_kk theta)_c
    lap = mad(rdx, half_cell_cond(gx, p.rdx[i - 1] * s_th[p.mat[o - 1]].k) * (th - t.theta[o - 1]), lap);
    lap = mad(rdx, half_cell_cond(gx, p.rdx[i + 1] * s_th[p.mat[o + 1]].k) * (th - t.theta[o + 1]), lap);
    lap = mad(rdy, half_cell_cond(gy, p.rdy[j - 1] * s_th[p.mat[o - PX]].k) * (th - t.theta[o - PX]), lap);
    lap = mad(rdy, half_cell_cond(gy, p.rdy[j + 1] * s_th[p.mat[o + PX]].k) * (th - t.theta[o + PX]), lap);
    lap = mad(rdz, half_cell_cond(gz, p.rdz[k - 1] * s_th[p.mat[o - PXY]].k) * (th - t.theta[o - PXY]), lap);
    lap = mad(rdz, half_cell_cond(gz, p.rdz[k + 1] * s_th[p.mat[o + PXY]].k) * (th - t.theta[o + PXY]), lap);
    const R thn = th - p.dt * me.irc * lap + dq * me.irc;
    t.theta_n[o] = thn;
    t.sig[o] = me.sigma0 * rcp<R>(thermal_den(me.alpha, thn));
}

// Conduction half of eq. (5) for the coupled sweep: theta_d = theta^n - dt/(rho c_p) (M_kk theta^n), all cells, into the
// other theta buffer (the sweep then adds the Joule heat of the step in place).  A thread owns V = 16 B / sizeof(R)
// consecutive cells in x: 128-bit loads of the centre, the +-y and +-z neighbour vectors, V + 1 x-face conductances
// shared between neighbouring cells.  Vectors past nx only touch pad cells (k = 0, theta = 0) and are not stored.
template <typename R>
__global__ void __launch_bounds__(256) k_diffuse(DevParams<R> p, const ThEntry<R> *ttable, const R *theta, R *theta_d) {
    constexpr int V = 16 / sizeof(R);
    struct alignas(16) VR { R v[V]; };
    const ThEntry<R> *s_th = ttable;       // a few 16/32-B entries: read through L1, no shared-memory copy and no barrier
    const int i0 = (blockIdx.x * blockDim.x + threadIdx.x) * V;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i0 >= p.nx || j >= p.ny) return;
    const long long PX = p.PX, PXY = p.PXY;
    const long long o = ((long long)k * p.PY + j) * PX + i0;
    auto ldv = [&](long long off) -> VR { return *reinterpret_cast<const VR *>(theta + off); };
    const VR th = ldv(o), tym = ldv(o - PX), typ = ldv(o + PX), tzm = ldv(o - PXY), tzp = ldv(o + PXY);
    const R txm = theta[o - 1], txp = theta[o + V];
    const R rdy = p.rdy[j], rdz = p.rdz[k];
    const R rdym = p.rdy[j - 1], rdyp = p.rdy[j + 1], rdzm = p.rdz[k - 1], rdzp = p.rdz[k + 1];
    // the V material ids of a vector as one aligned word (i0 is a multiple of V and the array origin is 128-B aligned)
    using IdT = typename std::conditional<V == 4, unsigned, unsigned short>::type;
    auto ldid = [&](long long off) -> unsigned { return *reinterpret_cast<const IdT *>(p.mat + off); };
    const unsigned idc = ldid(o), idym = ldid(o - PX), idyp = ldid(o + PX), idzm = ldid(o - PXY), idzp = ldid(o + PXY);
    const unsigned idl = p.mat[o - 1], idr = p.mat[o + V];
    // One material over the whole 7-point neighbourhood of the vector (the common case): the series conductance of two
    // equal half cells is k * 2/(d + d') = k / d~, i.e. k times the dual-length reciprocals the E update already uses.
    const unsigned rep_id = (idc & 0xffu) * (V == 4 ? 0x01010101u : 0x0101u);
    if (idc == rep_id && idym == rep_id && idyp == rep_id && idzm == rep_id && idzp == rep_id &&
        idl == (idc & 0xffu) && idr == (idc & 0xffu) && i0 + V <= p.nx) {
        const ThEntry<R> me = s_th[idc & 0xffu];
        const R cy0 = rdy * p.rty[j], cy1 = rdy * p.rty[j + 1], cz0 = rdz * p.rtz[k], cz1 = rdz * p.rtz[k + 1];
        const R scale = p.dt * me.irc * me.k;
        const VR rdxv = *reinterpret_cast<const VR *>(p.rdx + i0), rtxv = *reinterpret_cast<const VR *>(p.rtx + i0);
        const R rtxe = p.rtx[i0 + V];
        VR out;
#pragma unroll
        for (int c = 0; c < V; ++c) {
            const R t0 = th.v[c];
            const R tl = c > 0 ? th.v[c > 0 ? c - 1 : 0] : txm, tr = c < V - 1 ? th.v[c < V - 1 ? c + 1 : c] : txp;
            const R rtx1 = c < V - 1 ? rtxv.v[c < V - 1 ? c + 1 : c] : rtxe;
            R lap = rdxv.v[c] * (rtxv.v[c] * (t0 - tl) + rtx1 * (t0 - tr));
            lap = mad(cy0, t0 - tym.v[c], lap); lap = mad(cy1, t0 - typ.v[c], lap);
            lap = mad(cz0, t0 - tzm.v[c], lap); lap = mad(cz1, t0 - tzp.v[c], lap);
            out.v[c] = mad(-scale, lap, t0);
        }
        *reinterpret_cast<VR *>(theta_d + o) = out;
        return;
    }
    R kc[V + 2], rdx[V + 2];                                  // cells i0-1 .. i0+V
    kc[0] = s_th[idl].k; kc[V + 1] = s_th[idr].k;
#pragma unroll
    for (int c = 0; c < V; ++c) kc[c + 1] = s_th[(idc >> (8 * c)) & 0xff].k;
#pragma unroll
    for (int c = 0; c < V + 2; ++c) rdx[c] = p.rdx[i0 + c - 1];
    R gxf[V + 1];                                             // x faces between cells c-1 and c (c = 0 .. V)
#pragma unroll
    for (int c = 0; c < V + 1; ++c) gxf[c] = half_cell_cond(rdx[c] * kc[c], rdx[c + 1] * kc[c + 1]);
    VR out;
#pragma unroll
    for (int c = 0; c < V; ++c) {
        const R kme = kc[c + 1], t0 = th.v[c];
        const R gy = rdy * kme, gz = rdz * kme;
        const R tl = c > 0 ? th.v[c > 0 ? c - 1 : 0] : txm, tr = c < V - 1 ? th.v[c < V - 1 ? c + 1 : c] : txp;
        R lap = rdx[c + 1] * (gxf[c] * (t0 - tl) + gxf[c + 1] * (t0 - tr));
        lap = mad(rdy, half_cell_cond(gy, rdym * s_th[(idym >> (8 * c)) & 0xff].k) * (t0 - tym.v[c]), lap);
        lap = mad(rdy, half_cell_cond(gy, rdyp * s_th[(idyp >> (8 * c)) & 0xff].k) * (t0 - typ.v[c]), lap);
        lap = mad(rdz, half_cell_cond(gz, rdzm * s_th[(idzm >> (8 * c)) & 0xff].k) * (t0 - tzm.v[c]), lap);
        lap = mad(rdz, half_cell_cond(gz, rdzp * s_th[(idzp >> (8 * c)) & 0xff].k) * (t0 - tzp.v[c]), lap);
        out.v[c] = t0 - p.dt * s_th[(idc >> (8 * c)) & 0xff].irc * lap;
    }
    if (i0 + V <= p.nx) {
        *reinterpret_cast<VR *>(theta_d + o) = out;
    } else {
        for (int c = 0; c < V && i0 + c < p.nx; ++c) theta_d[o + c] = out.v[c];
    }
}

// ---- NODAL thermal stage: the paper's placement of T (7 092 878 thermal unknowns = the mesh nodes; eq.
// (4)-(6) L84-L96, M_kk = V0a^T D_k V0 L86; readings N1-N4 of DESIGN.md section 9; em_grid.thermal = 2, split kernels) ------
// a4 with the per-cell sigma(T^n): q_c += dt sigma_c / 16 sum_12 (E' + E)^2 (the Joule map stays per cell, C7)
template <typename R>
__global__ void __launch_bounds__(256) k_joule_sig(DevParams<R> p, const R *sig) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= p.nx || j >= p.ny) return;
    const long long PX = p.PX, PXY = p.PXY;
    const long long o = ((long long)k * p.PY + j) * PX + i;
    const R sg = sig[o];
    if (sg == R(0)) return;
    R s = 0;
#define EM_ACC(c, off) { const R t_ = p.Hn[c][o + (off)]; s = mad(t_, t_, s); }      /* E' + E as k_split_e_sig formed it */
    EM_ACC(0, 0) EM_ACC(0, PX) EM_ACC(0, PXY) EM_ACC(0, PXY + PX)
    EM_ACC(1, 0) EM_ACC(1, 1)  EM_ACC(1, PXY) EM_ACC(1, PXY + 1)
    EM_ACC(2, 0) EM_ACC(2, 1)  EM_ACC(2, PX)  EM_ACC(2, PX + 1)
#undef EM_ACC
    p.q[o] = mad(p.dt * sg * R(0.0625), s, p.q[o]);
}

// eq. (5) on the nodes.  One thread per node n = (i, j, k):
//   C_n theta_n' = C_n theta_n - dt sum_{e at n} (k_e A~_e / l_e) (theta_n - theta_m) + 1/2 sum_{e at n} dQ_e
//   k_e A~_e = sum over the <= 4 cells round e of k_c A_{c,e} / 4,   dQ_e = dt Ebar_e^2 l_e sum_c sigma_c(T^n) A_{c,e} / 4,
//   C_n = sum over the <= 8 cells round n of rho c_p V_c / 8.
// Cells outside the grid contribute nothing by themselves: their table entries hold k = 0 and 1/(rho c_p) = 0, their
// sigma(T) is 0 and their sizes read as 0 (vx, vy, vz are the cell sizes in fp64, length nx, ny, nz).
template <typename R>
__global__ void __launch_bounds__(256) k_thermal_nodal(DevParams<R> p, ThermalParams<R> t, const double *vx, const double *vy, const double *vz) {
    __shared__ ThEntry<R> s_th[kMaxTable];
    {
        const int tid = threadIdx.y * blockDim.x + threadIdx.x, nth = blockDim.x * blockDim.y;
        for (int m = tid; m < p.n_table; m += nth) s_th[m] = t.ttable[m];
        __syncthreads();
    }
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i > p.nx || j > p.ny) return;
    const long long PX = p.PX, PXY = p.PXY;
    const long long o = ((long long)k * p.PY + j) * PX + i;
    const long long stride[3] = {1, PX, PXY};
    const int node[3] = {i, j, k}, n[3] = {p.nx, p.ny, p.nz};
    const double *vv[3] = {vx, vy, vz};
    auto size = [&](int a, int c) -> R { return (c >= 0 && c < n[a]) ? (R)vv[a][c] : R(0); };
    // sizes of the two cell layers below (index 0) and above (1) the node along every axis
    R d[3][2];
#pragma unroll
    for (int a = 0; a < 3; ++a) { d[a][0] = size(a, node[a] - 1); d[a][1] = size(a, node[a]); }
    const R th0 = t.theta[o];
    R out = R(0), heat = R(0), cap = R(0);
#pragma unroll
    for (int a = 0; a < 3; ++a) {                        // edges along axis a; b, c: the two transverse axes
        const int b = (a + 1) % 3, c = (a + 2) % 3;
#pragma unroll
        for (int side = 0; side < 2; ++side) {           // the edge below (0) / above (1) the node
            const R len = d[a][side];
            if (len == R(0)) continue;
            const long long oe = side ? o : o - stride[a];                       // the edge is indexed by its lower node
            const long long om = side ? o + stride[a] : o - stride[a];           // the node at its other end
            R ka = R(0), sa = R(0);                                               // sum k_c A / 4, sum sigma_c A / 4
#pragma unroll
            for (int sb = 0; sb < 2; ++sb)
#pragma unroll
                for (int sc = 0; sc < 2; ++sc) {
                    const R area = d[b][sb] * d[c][sc] * R(0.25);
                    if (area == R(0)) continue;
                    const long long oc = oe - (sb ? 0 : stride[b]) - (sc ? 0 : stride[c]);   // cell (edge cell along a, b - 1 + sb, c - 1 + sc)
                    ka = mad(s_th[p.mat[oc]].k, area, ka);
                    sa = mad(t.sig[oc], area, sa);
                }
            out = mad(ka * rcp<R>(len), th0 - t.theta[om], out);
            const R eb = R(0.5) * p.Hn[a][oe];                                    // (E' + E) / 2 as k_split_e_sig formed it
            heat = mad(R(0.5) * p.dt * eb * eb * len, sa, heat);
        }
    }
#pragma unroll
    for (int sa_ = 0; sa_ < 2; ++sa_)
#pragma unroll
        for (int sb = 0; sb < 2; ++sb)
#pragma unroll
            for (int sc = 0; sc < 2; ++sc) {
                const R vol = d[0][sa_] * d[1][sb] * d[2][sc] * R(0.125);
                if (vol == R(0)) continue;
                const long long oc = o - (sa_ ? 0 : 1) - (sb ? 0 : PX) - (sc ? 0 : PXY);
                const R irc = s_th[p.mat[oc]].irc;
                if (irc > R(0)) cap = mad(rcp<R>(irc), vol, cap);
            }
    t.theta_n[o] = cap > R(0) ? th0 + (heat - p.dt * out) * rcp<R>(cap) : th0;
}

// eq. (6) per cell with the mean of the cell's 8 node temperatures (N4); cell layers k0 .. k0 + gridDim.z - 1
template <typename R>
__global__ void __launch_bounds__(256) k_sigma_nodal(DevParams<R> p, ThermalParams<R> t, int k0) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = k0 + blockIdx.z;
    if (i >= p.nx || j >= p.ny) return;
    const long long PX = p.PX, PXY = p.PXY;
    const long long o = ((long long)k * p.PY + j) * PX + i;
    const ThEntry<R> me = t.ttable[p.mat[o]];
    const R m = ((t.theta[o] + t.theta[o + 1]) + (t.theta[o + PX] + t.theta[o + PX + 1])) +
                ((t.theta[o + PXY] + t.theta[o + PXY + 1]) + (t.theta[o + PXY + PX] + t.theta[o + PXY + PX + 1]));
    t.sig[o] = me.sigma0 * rcp<R>(thermal_den(me.alpha, R(0.125) * m));
}

// z-slab halo of the nodal stage: the temperature rise of node plane kp, dense [(ny+1) x (nx+1)], out of (unpack = 0) or
// into (1) the padded array.  (The tangential E of the plane travels in k_pack_halo / k_unpack_halo as for every context.)
template <typename R>
__global__ void __launch_bounds__(256) k_node_plane(DevParams<R> p, R *theta, int kp, R *packed, int unpack) {
    const long long n = (long long)(p.ny + 1) * (p.nx + 1);
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    const int j = (int)(t / (p.nx + 1)), i = (int)(t % (p.nx + 1));
    const long long o = ((long long)kp * p.PY + j) * p.PX + i;
    if (unpack) theta[o] = packed[t]; else packed[t] = theta[o];
}

// sigma = sigma_0 / (1 + alpha theta) on every cell (after em_set_thermal / em_set_temperature_rise / em_reset)
template <typename R>
__global__ void __launch_bounds__(256) k_sigma_refresh(DevParams<R> p, ThermalParams<R> t) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= p.nx || j >= p.ny) return;
    const long long o = ((long long)k * p.PY + j) * p.PX + i;
    const ThEntry<R> me = t.ttable[p.mat[o]];
    // the expression of the stepping kernels, so that sigma(T) restored from theta (em_set_temperature_rise: resume of a
    // checkpoint, slab halos) has the bits the uninterrupted run holds
    t.sig[o] = me.sigma0 * rcp<R>(thermal_den(me.alpha, t.theta[o]));
}

// p_c = sigma_c(T) * 1/4 sum_12 (E_e)^2 with the CURRENT conductivity (PAPER.md L86 with eq. (6))
template <typename R>
__global__ void __launch_bounds__(256) k_power_sig(DevParams<R> p, const R *sig, R *out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= p.nx || j >= p.ny) return;
    const long long PX = p.PX, PXY = p.PXY;
    const long long o = ((long long)k * p.PY + j) * PX + i;
    R s = 0;
#define EM_SQ(c, off) { const R t_ = p.E[c][o + (off)]; s = mad(t_, t_, s); }
    EM_SQ(0, 0) EM_SQ(0, PX) EM_SQ(0, PXY) EM_SQ(0, PXY + PX)
    EM_SQ(1, 0) EM_SQ(1, 1)  EM_SQ(1, PXY) EM_SQ(1, PXY + 1)
    EM_SQ(2, 0) EM_SQ(2, 1)  EM_SQ(2, PX)  EM_SQ(2, PX + 1)
#undef EM_SQ
    out[((long long)k * p.ny + j) * p.nx + i] = sig[o] * R(0.25) * s;
}

}  // namespace em
