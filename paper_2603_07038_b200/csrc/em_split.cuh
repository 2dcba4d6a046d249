// em_split.cuh -- the "split" kernel strategy: one H-update kernel, one E-update kernel, one
// source kernel and one Joule kernel per time step (EM_KERNEL_SPLIT).  One thread per node/cell,
// neighbours through L1/L2.  This is the simple first CUDA path: it moves ~26 words per cell-update
// and exists for cross-checking the fused sweep (em_fused.cuh) and for grids too small to tile.
//
// Arithmetic (identical in both strategies):
//   a1  H' = H - nbar * (C_e E)            nbar = length-weighted mean of dt/mu over the 2 cells
//   a2  E' = E + r * (C_h H' - sigma_bar E)   r = loss coefficient of the area-weighted eps, sigma
//       (incremental form of ca E + cb C_h H', ca = 1 - sigma_bar r; masked to 0 on PEC-fixed edges)
//   a3  E' -= r * J                        on the source edges
//   a4  q_c += dt sigma_c / 16 * sum_12 (E' + E)^2
#pragma once
#include "em_common.cuh"

namespace em {

template <typename R>
__device__ __forceinline__ void load_table(MatEntry<R> *s_tab, const DevParams<R> &p) {
    const int tid = threadIdx.y * blockDim.x + threadIdx.x;
    const int nth = blockDim.x * blockDim.y;
    for (int t = tid; t < p.n_table; t += nth) s_tab[t] = p.table[t];
    __syncthreads();
}

// a1 -- PAPER.md L65 (S = curl mu^-1 curl, inner factor), SURVEY.md 8(c) a1.
template <typename R>
__global__ void __launch_bounds__(256) k_split_h(DevParams<R> p) {
    __shared__ MatEntry<R> s_tab[kMaxTable];
    load_table(s_tab, p);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i > p.nx || j > p.ny) return;
    const long long o = ((long long)k * p.PY + j) * p.PX + i;
    const long long PX = p.PX, PXY = p.PXY;
    const R ex = p.E[0][o], exj = p.E[0][o + PX], exk = p.E[0][o + PXY];
    const R ey = p.E[1][o], eyi = p.E[1][o + 1], eyk = p.E[1][o + PXY];
    const R ez = p.E[2][o], ezi = p.E[2][o + 1], ezj = p.E[2][o + PX];
    const R n0 = s_tab[p.mat[o]].n;
    const R nxm = s_tab[p.mat[o - 1]].n, nym = s_tab[p.mat[o - PX]].n, nzm = s_tab[p.mat[o - PXY]].n;
    const R nbx = lerp(nxm, n0, p.fx[i]), nby = lerp(nym, n0, p.fy[j]), nbz = lerp(nzm, n0, p.fz[k]);
    const R rdx = p.rdx[i], rdy = p.rdy[j], rdz = p.rdz[k];
    p.H[0][o] -= nbx * ((ezj - ez) * rdy - (eyk - ey) * rdz);
    p.H[1][o] -= nby * ((exk - ex) * rdz - (ezi - ez) * rdx);
    p.H[2][o] -= nbz * ((eyi - ey) * rdx - (exj - ex) * rdy);
}

// Edge coefficients (r, sigma_bar) of the three edges at node (i,j,k) from the 7 surrounding cells, and h2 = 2 - r sigma_bar
// formed WITHOUT cancellation (CD: 2 (eps/dt) r): E' + E = r (C_h H' - J) + h2 E is what the Joule sum needs, and in a good
// conductor (CD: E' = -E + small) adding the stored E' and E instead loses the digits in fp32.
template <typename R, int LOSS>
__device__ __forceinline__ void edge_coeffs(const MatEntry<R> *tab, const uint8_t *mat, long long o,
                                            long long PX, long long PXY, R fx, R fy, R fz,
                                            R r[3], R sg[3], R h2[3]) {
    const MatEntry<R> c000 = tab[mat[o]], c100 = tab[mat[o - 1]], c010 = tab[mat[o - PX]];
    const MatEntry<R> c110 = tab[mat[o - PX - 1]], c001 = tab[mat[o - PXY]];
    const MatEntry<R> c101 = tab[mat[o - PXY - 1]], c011 = tab[mat[o - PXY - PX]];
    // Ex: cells (i, j-1..j, k-1..k)
    {
        const R A = lerp(lerp(c011.a, c001.a, fy), lerp(c010.a, c000.a, fy), fz);
        const R B = lerp(lerp(c011.b, c001.b, fy), lerp(c010.b, c000.b, fy), fz);
        const R m = (c011.m * c001.m) * (c010.m * c000.m);
        const R rr = loss_r<R, LOSS>(A, B);
        r[0] = m * rr; sg[0] = B; h2[0] = (LOSS == 0) ? R(2) * A * rr : R(2) - rr * B;
    }
    // Ey: cells (i-1..i, j, k-1..k)
    {
        const R A = lerp(lerp(c101.a, c001.a, fx), lerp(c100.a, c000.a, fx), fz);
        const R B = lerp(lerp(c101.b, c001.b, fx), lerp(c100.b, c000.b, fx), fz);
        const R m = (c101.m * c001.m) * (c100.m * c000.m);
        const R rr = loss_r<R, LOSS>(A, B);
        r[1] = m * rr; sg[1] = B; h2[1] = (LOSS == 0) ? R(2) * A * rr : R(2) - rr * B;
    }
    // Ez: cells (i-1..i, j-1..j, k)
    {
        const R A = lerp(lerp(c110.a, c010.a, fx), lerp(c100.a, c000.a, fx), fy);
        const R B = lerp(lerp(c110.b, c010.b, fx), lerp(c100.b, c000.b, fx), fy);
        const R m = (c110.m * c010.m) * (c100.m * c000.m);
        const R rr = loss_r<R, LOSS>(A, B);
        r[2] = m * rr; sg[2] = B; h2[2] = (LOSS == 0) ? R(2) * A * rr : R(2) - rr * B;
    }
}

// a2 -- PAPER.md eq. (2)-(3) L69-L76 in leapfrog form; reads E, writes En.
template <typename R, int LOSS>
__global__ void __launch_bounds__(256) k_split_e(DevParams<R> p) {
    __shared__ MatEntry<R> s_tab[kMaxTable];
    load_table(s_tab, p);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i > p.nx || j > p.ny) return;
    const long long PX = p.PX, PXY = p.PXY;
    const long long o = ((long long)k * p.PY + j) * PX + i;
    R r[3], sg[3], h2[3];
    edge_coeffs<R, LOSS>(s_tab, p.mat, o, PX, PXY, p.fx[i], p.fy[j], p.fz[k], r, sg, h2);
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
    // E' + E for the Joule kernels, in the arrays the split strategy does not use otherwise (H is updated in place)
    p.Hn[0][o] = mad(r[0], cx, h2[0] * ex);
    p.Hn[1][o] = mad(r[1], cy, h2[1] * ey);
    p.Hn[2][o] = mad(r[2], cz, h2[2] * ez);
}

// a4 -- PAPER.md L86 (P = D_sigma e^2), SURVEY.md 8(c) a4/C7 (time-centred, cell-centred).
template <typename R>
__global__ void __launch_bounds__(256) k_split_joule(DevParams<R> p) {
    __shared__ MatEntry<R> s_tab[kMaxTable];
    load_table(s_tab, p);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= p.nx || j >= p.ny) return;
    const long long PX = p.PX, PXY = p.PXY;
    const long long o = ((long long)k * p.PY + j) * PX + i;
    const R sig = s_tab[p.mat[o]].b;
    if (sig == R(0)) return;                    // sigma_c = 0: q_c never changes
    R s = 0;
#define EM_ACC(c, off) { const R t_ = p.Hn[c][o + (off)]; s = mad(t_, t_, s); }      /* E' + E as k_split_e formed it */
    EM_ACC(0, 0) EM_ACC(0, PX) EM_ACC(0, PXY) EM_ACC(0, PXY + PX)
    EM_ACC(1, 0) EM_ACC(1, 1)  EM_ACC(1, PXY) EM_ACC(1, PXY + 1)
    EM_ACC(2, 0) EM_ACC(2, 1)  EM_ACC(2, PX)  EM_ACC(2, PX + 1)
#undef EM_ACC
    p.q[o] = mad(p.dt * sig * R(0.0625), s, p.q[o]);
}

}  // namespace em
