// em_aux.cuh -- setup / output kernels around the hot path: PEC masking after em_set_field,
// source coefficients and injection (a3), power-density map, fp64 Joule total, probe gather.
#pragma once
#include "em_common.cuh"
#include "em_split.cuh"

namespace em {

// Source lists on the device.  "Unique edge" u owns contributions [cbeg[u], cbeg[u+1]) so that
// overlapping ports add in a fixed order.
template <typename R>
struct DevSources {
    int n_unique;
    const long long *off;     // padded offset of the edge
    const int *comp;          // 0,1,2
    R *r;                     // loss coefficient r_e of the edge (filled by k_source_coef)
    const int *cbeg;          // n_unique + 1
    const int *con_port;      // per contribution
    const R *con_scale;       // amplitude * weight
    const long long *port_woff, *port_wlen;
    const R *wave;
};

// PMC walls: a pad cell that lies beyond PMC walls ONLY gets the id of the
// "outside / PMC" table entry (mask 1, zero weight in every mean because the pad spacings are 0), so the
// tangential E of a PMC wall stays an unknown; pad cells beyond any PEC wall keep the mask-0 entry.
// base = the element (i, j, k) = (-1, -1, -1); n = PX * PY * PZ elements; pmc_mask bit b = wall b is PMC.
__global__ void __launch_bounds__(256) k_pad_pmc(uint8_t *base, int nx, int ny, int nz, int PX, int PY, long long n,
                                                 int pmc_mask, uint8_t pmc_id) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    const long long PXY = (long long)PX * PY;
    const int k = (int)(t / PXY) - 1;
    const long long rem = t % PXY;
    const int j = (int)(rem / PX) - 1, i = (int)(rem % PX) - 1;
    int beyond = 0;                                   // walls this cell lies beyond
    if (i < 0) beyond |= 1; if (i >= nx) beyond |= 2;
    if (j < 0) beyond |= 4; if (j >= ny) beyond |= 8;
    if (k < 0) beyond |= 16; if (k >= nz) beyond |= 32;
    if (beyond != 0 && (beyond & ~pmc_mask) == 0) base[t] = pmc_id;
}

// Zero the edge array `e` of direction comp wherever the edge is PEC-fixed (mask product of its 4 cells is 0).
template <typename R>
__global__ void __launch_bounds__(256) k_mask_fixed(DevParams<R> p, R *e, int comp, int k0) {
    __shared__ MatEntry<R> s_tab[kMaxTable];
    load_table(s_tab, p);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z + k0;
    if (i > p.nx || j > p.ny) return;
    const long long PX = p.PX, PXY = p.PXY;
    const long long o = ((long long)k * p.PY + j) * PX + i;
    const uint8_t *mat = p.mat;
    R m;
    if (comp == 0)      m = s_tab[mat[o]].m * s_tab[mat[o - PX]].m * s_tab[mat[o - PXY]].m * s_tab[mat[o - PXY - PX]].m;
    else if (comp == 1) m = s_tab[mat[o]].m * s_tab[mat[o - 1]].m * s_tab[mat[o - PXY]].m * s_tab[mat[o - PXY - 1]].m;
    else                m = s_tab[mat[o]].m * s_tab[mat[o - 1]].m * s_tab[mat[o - PX]].m * s_tab[mat[o - PX - 1]].m;
    if (m == R(0)) e[o] = R(0);
}

// Halo of a z-slab decomposition: the tangential E of node plane kp, packed [Ex (ny+1) x nx | Ey ny x (nx+1)],
// and -- thermally coupled contexts -- the temperature rise of cell layer kl behind it [ny x nx].  One kernel each way.
template <typename R>
__global__ void __launch_bounds__(256) k_pack_halo(DevParams<R> p, const R *ex, const R *ey, const R *theta, int kp, int kl, R *dst) {
    const long long n0 = (long long)(p.ny + 1) * p.nx, n1 = (long long)p.ny * (p.nx + 1), n2 = theta ? (long long)p.ny * p.nx : 0;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n0) {
        const int j = (int)(t / p.nx), i = (int)(t % p.nx);
        dst[t] = ex[((long long)kp * p.PY + j) * p.PX + i];
    } else if (t < n0 + n1) {
        const long long u = t - n0;
        const int j = (int)(u / (p.nx + 1)), i = (int)(u % (p.nx + 1));
        dst[t] = ey[((long long)kp * p.PY + j) * p.PX + i];
    } else if (t < n0 + n1 + n2) {
        const long long u = t - n0 - n1;
        const int j = (int)(u / p.nx), i = (int)(u % p.nx);
        dst[t] = theta[((long long)kl * p.PY + j) * p.PX + i];
    }
}

// The reverse: PEC-fixed edges of the plane stay 0 (the mask product of the edge's four cells, as in k_mask_fixed); the
// temperature rise goes into the layer and sigma(T) of the layer's cells is refreshed in both sigma buffers (eq. (6)).
template <typename R>
__global__ void __launch_bounds__(256) k_unpack_halo(DevParams<R> p, R *ex, R *ey, R *theta, R *sig_a, R *sig_b,
                                                     const ThEntry<R> *ttable, int kp, int kl, const R *src) {
    __shared__ MatEntry<R> s_tab[kMaxTable];
    load_table(s_tab, p);
    const long long n0 = (long long)(p.ny + 1) * p.nx, n1 = (long long)p.ny * (p.nx + 1), n2 = theta ? (long long)p.ny * p.nx : 0;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long PX = p.PX, PXY = p.PXY;
    const uint8_t *mat = p.mat;
    if (t < n0) {
        const int j = (int)(t / p.nx), i = (int)(t % p.nx);
        const long long o = ((long long)kp * p.PY + j) * PX + i;
        const R m = s_tab[mat[o]].m * s_tab[mat[o - PX]].m * s_tab[mat[o - PXY]].m * s_tab[mat[o - PXY - PX]].m;
        ex[o] = m == R(0) ? R(0) : src[t];
    } else if (t < n0 + n1) {
        const long long u = t - n0;
        const int j = (int)(u / (p.nx + 1)), i = (int)(u % (p.nx + 1));
        const long long o = ((long long)kp * p.PY + j) * PX + i;
        const R m = s_tab[mat[o]].m * s_tab[mat[o - 1]].m * s_tab[mat[o - PXY]].m * s_tab[mat[o - PXY - 1]].m;
        ey[o] = m == R(0) ? R(0) : src[t];
    } else if (t < n0 + n1 + n2) {
        const long long u = t - n0 - n1;
        const int j = (int)(u / p.nx), i = (int)(u % p.nx);
        const long long o = ((long long)kl * p.PY + j) * PX + i;
        const ThEntry<R> me = ttable[mat[o]];
        const R th = src[t];
        theta[o] = th;
        const R sg = me.sigma0 * rcp<R>(thermal_den(me.alpha, th));     // the expression of the stepping kernels (bit-identical slabs)
        sig_a[o] = sg; sig_b[o] = sg;
    }
}

// r_e for every unique source edge; flags[u] = 1 if the edge is PEC-fixed (argument error).
template <typename R, int LOSS>
__global__ void k_source_coef(DevParams<R> p, DevSources<R> s, int *fixed_flags) {
    const int u = blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= s.n_unique) return;
    const long long o = s.off[u];
    const long long PX = p.PX, PXY = p.PXY;
    const long long kk = o / PXY, rem = o - kk * PXY;   // o >= 0 for in-range edges
    const int j = (int)(rem / PX), i = (int)(rem - (long long)j * PX), k = (int)kk;
    R r[3], sg[3], h2[3];
    edge_coeffs<R, LOSS>(p.table, p.mat, o, PX, PXY, p.fx[i], p.fy[j], p.fz[k], r, sg, h2);
    const R re = r[s.comp[u]];
    s.r[u] = re;
    fixed_flags[u] = (re == R(0)) ? 1 : 0;
}

// a3 -- E^{n+1} -= r_e * J_e^{n+1/2}   ("-dt^2 (dJ/dt)^n")
// (t0..t2: the E' + E arrays of the split strategy, which carry the same -r_e J)
template <typename R>
__global__ void k_apply_source(R *e0, R *e1, R *e2, R *t0, R *t1, R *t2, DevSources<R> s, long long step) {
    const int u = blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= s.n_unique) return;
    R J = 0;
    for (int c = s.cbeg[u]; c < s.cbeg[u + 1]; ++c) {
        const int pt = s.con_port[c];
        if (step < s.port_wlen[pt]) J = mad(s.con_scale[c], s.wave[s.port_woff[pt] + step], J);
    }
    R *e = s.comp[u] == 0 ? e0 : (s.comp[u] == 1 ? e1 : e2);
    e[s.off[u]] = mad(-s.r[u], J, e[s.off[u]]);
    R *t = s.comp[u] == 0 ? t0 : (s.comp[u] == 1 ? t1 : t2);
    t[s.off[u]] = mad(-s.r[u], J, t[s.off[u]]);
}

// p_c = sigma_c * 1/4 sum_12 (E_e)^2 into a dense [nz][ny][nx] map
template <typename R>
__global__ void __launch_bounds__(256) k_power(DevParams<R> p, R *out) {
    __shared__ MatEntry<R> s_tab[kMaxTable];
    load_table(s_tab, p);
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
    out[((long long)k * p.ny + j) * p.nx + i] = s_tab[p.mat[o]].b * R(0.25) * s;
}

// Q = sum_c q_c V_c in fp64, fixed order: per-block partials then one block.
template <typename R>
__global__ void __launch_bounds__(256) k_energy_partial(DevParams<R> p, const double *vx, const double *vy,
                                                        const double *vz, int k0, int k1, double *partial) {
    __shared__ double sh[256];
    const long long ncell = (long long)p.nx * p.ny * (k1 - k0);           // cell layers k0 <= k < k1
    double acc = 0.0;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < ncell; c += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(c % p.nx); const long long t = c / p.nx;
        const int j = (int)(t % p.ny); const int k = k0 + (int)(t / p.ny);
        acc += (double)p.q[((long long)k * p.PY + j) * p.PX + i] * (vx[i] * vy[j] * vz[k]);
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

__global__ void __launch_bounds__(256) k_energy_final(const double *partial, int n, double *out) {
    __shared__ double sh[256];
    double acc = 0.0;
    for (int c = threadIdx.x; c < n; c += 256) acc += partial[c];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0];
}

// em_check_finite: *flag = 1 if any of the n values is Inf or NaN (every thread that finds one stores the same 1)
template <typename R>
__global__ void __launch_bounds__(256) k_check_finite(const R *a, long long n, int *flag) {
    const R big = sizeof(R) == 4 ? (R)3.402823466e+38F : (R)1.7976931348623157e+308;
    bool bad = false;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x)
        bad = bad || !(::fabs(a[t]) <= big);
    if (bad) *flag = 1;
}

template <typename R>
struct ProbeArrays { const R *f[9]; };

template <typename R>
__global__ void k_probe(ProbeArrays<R> a, const long long *off, const int *comp, int n, double *out) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) out[t] = (double)a.f[comp[t]][off[t]];
}

}  // namespace em
