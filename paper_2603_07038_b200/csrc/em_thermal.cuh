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
                                                long long PX, long long PXY, R fx, R fy, R fz, R r[3], R sg[3]) {
    const MatEntry<R> c000 = tab[mat[o]], c100 = tab[mat[o - 1]], c010 = tab[mat[o - PX]];
    const MatEntry<R> c110 = tab[mat[o - PX - 1]], c001 = tab[mat[o - PXY]];
    const MatEntry<R> c101 = tab[mat[o - PXY - 1]], c011 = tab[mat[o - PXY - PX]];
    const R b000 = sig[o], b100 = sig[o - 1], b010 = sig[o - PX], b110 = sig[o - PX - 1];
    const R b001 = sig[o - PXY], b101 = sig[o - PXY - 1], b011 = sig[o - PXY - PX];
    {   // Ex: cells (i, j-1..j, k-1..k)
        const R A = lerp(lerp(c011.a, c001.a, fy), lerp(c010.a, c000.a, fy), fz);
        const R B = lerp(lerp(b011, b001, fy), lerp(b010, b000, fy), fz);
        const R m = (c011.m * c001.m) * (c010.m * c000.m);
        r[0] = m * loss_r<R, LOSS>(A, B); sg[0] = B;
    }
    {   // Ey: cells (i-1..i, j, k-1..k)
        const R A = lerp(lerp(c101.a, c001.a, fx), lerp(c100.a, c000.a, fx), fz);
        const R B = lerp(lerp(b101, b001, fx), lerp(b100, b000, fx), fz);
        const R m = (c101.m * c001.m) * (c100.m * c000.m);
        r[1] = m * loss_r<R, LOSS>(A, B); sg[1] = B;
    }
    {   // Ez: cells (i-1..i, j-1..j, k)
        const R A = lerp(lerp(c110.a, c010.a, fx), lerp(c100.a, c000.a, fx), fy);
        const R B = lerp(lerp(b110, b010, fx), lerp(b100, b000, fx), fy);
        const R m = (c110.m * c010.m) * (c100.m * c000.m);
        r[2] = m * loss_r<R, LOSS>(A, B); sg[2] = B;
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
    R r[3], sg[3];
    edge_coeffs_sig<R, LOSS>(s_tab, p.mat, sig, o, PX, PXY, p.fx[i], p.fy[j], p.fz[k], r, sg);
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
    R r[3], sg[3];
    edge_coeffs_sig<R, LOSS>(p.table, p.mat, sig, o, PX, PXY, p.fx[i], p.fy[j], p.fz[k], r, sg);
    s.r[u] = r[s.comp[u]];
}

// series conductance per unit face area of the two half cells: k_f / l~_f = 2 / (d_a/k_a + d_b/k_b) = 2 g_a g_b / (g_a + g_b)
// with the half-cell conductances g = k/d; 0 if either cell does not conduct (k = 0, or a pad cell: 1/d = 0)
template <typename R> __device__ __forceinline__ R half_cell_cond(R ga, R gb) {
    const R den = ga + gb;
    return den > R(0) ? R(2) * ga * gb * rcp<R>(den) : R(0);
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
#define EM_ACC(c, off) { const R t_ = p.En[c][o + (off)] + p.E[c][o + (off)]; s = mad(t_, t_, s); }
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
    t.sig[o] = me.sigma0 * rcp<R>(R(1) + me.alpha * thn);
}

// Conduction half of eq. (5) for the coupled sweep: theta_d = theta^n - dt/(rho c_p) (M_kk theta^n), all cells, into the
// other theta buffer (the sweep then adds the Joule heat of the step in place).
template <typename R>
__global__ void __launch_bounds__(256) k_diffuse(DevParams<R> p, const ThEntry<R> *ttable, const R *theta, R *theta_d) {
    __shared__ ThEntry<R> s_th[kMaxTable];
    {
        const int tid = threadIdx.y * blockDim.x + threadIdx.x, nth = blockDim.x * blockDim.y;
        for (int m = tid; m < p.n_table; m += nth) s_th[m] = ttable[m];
        __syncthreads();
    }
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= p.nx || j >= p.ny) return;
    const long long PX = p.PX, PXY = p.PXY;
    const long long o = ((long long)k * p.PY + j) * PX + i;
    const ThEntry<R> me = s_th[p.mat[o]];
    const R th = theta[o];
    const R rdx = p.rdx[i], rdy = p.rdy[j], rdz = p.rdz[k];
    const R gx = rdx * me.k, gy = rdy * me.k, gz = rdz * me.k;
    R lap = R(0);
    lap = mad(rdx, half_cell_cond(gx, p.rdx[i - 1] * s_th[p.mat[o - 1]].k) * (th - theta[o - 1]), lap);
    lap = mad(rdx, half_cell_cond(gx, p.rdx[i + 1] * s_th[p.mat[o + 1]].k) * (th - theta[o + 1]), lap);
    lap = mad(rdy, half_cell_cond(gy, p.rdy[j - 1] * s_th[p.mat[o - PX]].k) * (th - theta[o - PX]), lap);
    lap = mad(rdy, half_cell_cond(gy, p.rdy[j + 1] * s_th[p.mat[o + PX]].k) * (th - theta[o + PX]), lap);
    lap = mad(rdz, half_cell_cond(gz, p.rdz[k - 1] * s_th[p.mat[o - PXY]].k) * (th - theta[o - PXY]), lap);
    lap = mad(rdz, half_cell_cond(gz, p.rdz[k + 1] * s_th[p.mat[o + PXY]].k) * (th - theta[o + PXY]), lap);
    theta_d[o] = th - p.dt * me.irc * lap;
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
    t.sig[o] = me.sigma0 / (R(1) + me.alpha * t.theta[o]);
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
