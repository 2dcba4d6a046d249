/*
 * em_oracle.c -- plain, slow, obviously-correct CPU ORACLE of the EM time-marching hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load it.  It shares no code, header,
 * table or helper with the CUDA library under paper_2603_07038_b200/csrc and include/em.h.
 *
 * What it computes (all in fp64, dense logical arrays, triple loops, in the paper's order):
 *   the explicit central-difference update of the edge-based vector wave equation
 *       D_eps e'' + (D_sigma e)' + S e = -J'                       PAPER.md L63  eq. (1)
 *       M e^{n+1} = N e^n - K e^{n-1} - dt^2 (dJ/dt)^n             PAPER.md L69  eq. (2)
 *       M,K = D_eps +- dt/2 D_sigma,  N = 2 D_eps - dt^2 S         PAPER.md L73-L76 eq. (3)
 *   written as the algebraically identical first-order E/H leapfrog with S = C_h D_nu C_e
 *   (the equivalence is pinned by tests/test_oracle_dense.py, which iterates
 *   eq. (2)-(3) literally with dense matrices), plus the Joule heat P = D_sigma e^2
 *    accumulated per cell.
 *
 * Unknown placement (pinned by the DOF count of PAPER.md L160):
 *   Ex(i,j,k) i<nx, j<=ny, k<=nz : edge from node (i,j,k) to (i+1,j,k); Ey, Ez cyclic.
 *   Hx(i,j,k) i<=nx, j<ny, k<nz  : x-normal face at node plane i over cell (j,k); Hy, Hz cyclic.
 * Arrays are C-ordered [k][j][i], x fastest.
 *
 * Readings of the paper where it is silent are those of SURVEY.md 8(c) C1-C20 (listed in
 * DESIGN.md).  Pins: tests/test_oracle_*.py (TE101 closed form, energy conservation, Poynting
 * balance, divergence invariants, conductor decay + Joule geometric series, dense eq. (2)-(3)
 * brute force, worked impulse example, axis-permutation symmetry, CFL power iteration) and
 * tests/test_oracle_pmc.py for the PMC walls of PAPER.md L142 (mirror-image equivalence with the all-PEC
 * doubled domain, quarter-wave closed form, energy and Poynting balance with mixed walls, dense eq. (2)-(3)).
 * Thermal stage (NEXT-1: PAPER.md eq. (4)-(6)) -- emo_set_thermal & co. at the end of this file -- is pinned by
 * tests/test_oracle_thermal.py (adiabatic scalar recurrence + exact energy balance, cosine-mode diffusion closed form,
 * heat conservation == Joule energy, dense V0a^T D_k V0); its NODAL variant (the paper's placement of T, emo_set_thermal_nodal,
 * thermal_step_nodal) by tests/test_oracle_thermal_nodal.py (the paper's printed DOF count, the dense B^T diag(k A~/l) B
 * assembled cell by cell, the DCT-I cosine-mode decay, the adiabatic scalar recurrence with the wall nodes, heat gained ==
 * Joule energy per step).
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define EMO_OK 0
#define EMO_ERR_INVALID_ARG 1
#define EMO_ERR_UNSUPPORTED 5

#define EMO_LOSS_CD 0
#define EMO_LOSS_EXP 1
#define EMO_BC_PEC 0   /* tangential E held at 0 on the wall                                        */
#define EMO_BC_PMC 1   /* the paper's truncation: tangential H = 0 on the wall.  The
                          wall's tangential E edges stay unknowns; their dual face is the half face
                          inside the domain (dual length d/2) and H outside the domain is 0
                          (SURVEY.md 8(c) C8).  Equivalent to mirroring the domain in the wall
                          (tangential E even, tangential H odd), which is how the tests pin it. */

typedef struct {
    int32_t nx, ny, nz;
    const double *dx, *dy, *dz;   /* cell sizes, lengths nx, ny, nz */
    int32_t loss_mode;            /* EMO_LOSS_CD (paper eq. 3) or EMO_LOSS_EXP */
    int32_t bc[6];                /* -x,+x,-y,+y,-z,+z ; EMO_BC_PEC or EMO_BC_PMC */
} emo_grid;

typedef struct { double eps, mu, sigma; int32_t flags; } emo_material;   /* flags bit0 = PEC */
typedef struct { int64_t edge_begin, edge_end; double amplitude; int64_t wave_offset, wave_len; } emo_port;
typedef struct { int32_t comp, i, j, k; double weight; } emo_edge;
typedef struct { int32_t comp, i, j, k; } emo_probe_pt;

typedef struct emo_ctx {
    int32_t nx, ny, nz, loss_mode;
    int32_t bc[6];
    double dt;
    double *dx, *dy, *dz;          /* primal lengths */
    double *tx, *ty, *tz;          /* dual lengths d~ (nx+1, ny+1, nz+1) */
    uint8_t *mat;                  /* [nz][ny][nx] */
    double *sigma_c;               /* per-cell sigma: the table's, or sigma(T) of eq. (6) when thermal coupling is on */
    double *eps_c;                 /* per-cell eps (from the table) */
    uint8_t *pec_c;                /* per-cell PEC-material flag */
    /* thermal coupling (eq. (4)-(6), L84-L96; NEXT-1 of SURVEY.md 8(f)); off unless emo_set_thermal */
    int32_t thermal;               /* 0 off, 1 theta per CELL (readings T1-T5), 2 theta per NODE (the paper's placement, N1-N4) */
    double *theta, *theta_n;       /* temperature rise T - T0 per cell (thermal = 1) or per node (2), and the next level */
    double *dq;                    /* Joule energy density deposited in the current step [J/m^3] */
    double *sigma0_c, *rho_cp_c, *kth_c, *alpha_c;
    double *E[3], *H[3];           /* fields */
    double *En[3];                 /* E^{n+1} scratch */
    double *ca[3], *cb[3];         /* per-edge update coefficients (0,0 on fixed edges) */
    uint8_t *fixed[3];             /* 1 = PEC-fixed edge */
    double *nu[3];                 /* per-face 1/mu */
    double *J[3];                  /* source current density at t_{n+1/2} */
    double *q;                     /* accumulated Joule energy density [J/m^3], per cell */
    int64_t step;                  /* absolute step index n */
    int32_t n_ports; emo_port *ports; int64_t n_edges; emo_edge *edges; int64_t n_wave; double *wave;
} emo_ctx;

/* ---- logical array extents ---------------------------------------------------------------- */
static void dims_of(const emo_ctx *c, int comp, int *sx, int *sy, int *sz) {
    int nx = c->nx, ny = c->ny, nz = c->nz;
    switch (comp) {
    case 0: *sx = nx;     *sy = ny + 1; *sz = nz + 1; break;   /* Ex */
    case 1: *sx = nx + 1; *sy = ny;     *sz = nz + 1; break;   /* Ey */
    case 2: *sx = nx + 1; *sy = ny + 1; *sz = nz;     break;   /* Ez */
    case 3: *sx = nx + 1; *sy = ny;     *sz = nz;     break;   /* Hx */
    case 4: *sx = nx;     *sy = ny + 1; *sz = nz;     break;   /* Hy */
    default:*sx = nx;     *sy = ny;     *sz = nz + 1; break;   /* Hz */
    }
}
static int64_t count_of(const emo_ctx *c, int comp) {
    int sx, sy, sz; dims_of(c, comp, &sx, &sy, &sz); return (int64_t)sx * sy * sz;
}
#define IX(sx, sy, i, j, k) (((int64_t)(k) * (sy) + (j)) * (sx) + (i))
/* shorthand index macros for the six components */
#define EX(i,j,k) IX(nx,     ny + 1, i, j, k)
#define EY(i,j,k) IX(nx + 1, ny,     i, j, k)
#define EZ(i,j,k) IX(nx + 1, ny + 1, i, j, k)
#define HX(i,j,k) IX(nx + 1, ny,     i, j, k)
#define HY(i,j,k) IX(nx,     ny + 1, i, j, k)
#define HZ(i,j,k) IX(nx,     ny,     i, j, k)
#define CELL(i,j,k) IX(nx, ny, i, j, k)

int32_t emo_set_threads(int32_t n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
    return omp_get_max_threads();
#else
    (void)n; return 1;
#endif
}

/* CFL bound: min_c sqrt(eps mu)/sqrt(dx^-2 + dy^-2 + dz^-2) */
int32_t emo_cfl_dt(const emo_grid *g, const uint8_t *mat, const emo_material *tab, int32_t n_mat, double *dt_max) {
    if (!g || !mat || !tab || !dt_max) return EMO_ERR_INVALID_ARG;
    int nx = g->nx, ny = g->ny, nz = g->nz;
    double best = INFINITY;
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                int m = mat[CELL(i, j, k)];
                if (m >= n_mat) return EMO_ERR_INVALID_ARG;
                double s = sqrt(tab[m].eps * tab[m].mu);
                double gsum = 1.0 / (g->dx[i] * g->dx[i]) + 1.0 / (g->dy[j] * g->dy[j]) + 1.0 / (g->dz[k] * g->dz[k]);
                double v = s / sqrt(gsum);
                if (v < best) best = v;
            }
    *dt_max = best;
    return EMO_OK;
}

/* Loss coefficients for one edge (SURVEY.md 8(c) "Coefficients"; CD = PAPER.md eq. (3)). */
static void loss_coeff(int mode, double eps, double sig, double dt, double *ca, double *cb) {
    if (mode == EMO_LOSS_CD) {
        double m = eps / dt + 0.5 * sig;      /* M/dt   = D_eps/dt + D_sigma/2 */
        double kk = eps / dt - 0.5 * sig;     /* K/dt                             */
        *ca = kk / m;
        *cb = 1.0 / m;
    } else {
        if (sig > 0.0) {
            double u = sig * dt / eps;
            *ca = exp(-u);
            *cb = -expm1(-u) / sig;
        } else {
            *ca = 1.0;
            *cb = dt / eps;
        }
    }
}

static void free_ctx(emo_ctx *c) {
    if (!c) return;
    free(c->dx); free(c->dy); free(c->dz); free(c->tx); free(c->ty); free(c->tz);
    free(c->mat); free(c->sigma_c); free(c->q); free(c->eps_c); free(c->pec_c);
    free(c->theta); free(c->theta_n); free(c->dq); free(c->sigma0_c); free(c->rho_cp_c); free(c->kth_c); free(c->alpha_c);
    for (int a = 0; a < 3; ++a) {
        free(c->E[a]); free(c->H[a]); free(c->En[a]); free(c->ca[a]); free(c->cb[a]);
        free(c->fixed[a]); free(c->nu[a]); free(c->J[a]);
    }
    free(c->ports); free(c->edges); free(c->wave);
    free(c);
}

int32_t emo_destroy(emo_ctx *c) { free_ctx(c); return EMO_OK; }

/* D_eps, D_sigma on the edges (SURVEY.md 8(c) "Coefficients", C5) from the per-cell eps, sigma and PEC flags, and
 * the update coefficients ca, cb of every non-fixed edge.  Called once at create, and again after every step when
 * sigma depends on the temperature ("D_sigma(T^n) ... updated at each time step"). */
static void edge_coefficients(emo_ctx *c) {
    const int nx = c->nx, ny = c->ny, nz = c->nz;
    const int wx0 = c->bc[0] == EMO_BC_PEC, wx1 = c->bc[1] == EMO_BC_PEC, wy0 = c->bc[2] == EMO_BC_PEC,
              wy1 = c->bc[3] == EMO_BC_PEC, wz0 = c->bc[4] == EMO_BC_PEC, wz1 = c->bc[5] == EMO_BC_PEC;
    /* ---- D_eps, D_sigma on edges: area-weighted mean over the <=4 cells round the edge ------ */
    /* Ex(i,j,k): cells (i, j', k'), j' in {j-1,j}, k' in {k-1,k}, weight dy[j'] dz[k']            */
    for (int k = 0; k <= nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i < nx; ++i) {
        double sw = 0, se = 0, ss = 0; int pec = 0;
        for (int kk = k - 1; kk <= k; ++kk) for (int jj = j - 1; jj <= j; ++jj) {
            if (jj < 0 || jj >= ny || kk < 0 || kk >= nz) continue;
            const int64_t q = CELL(i, jj, kk);
            double w = c->dy[jj] * c->dz[kk];
            sw += w; se += w * c->eps_c[q]; ss += w * c->sigma_c[q]; pec |= c->pec_c[q];
        }
        int fx = (j == 0 && wy0) || (j == ny && wy1) || (k == 0 && wz0) || (k == nz && wz1) || pec;   /* PEC walls / PEC material */
        int64_t e = EX(i, j, k);
        c->fixed[0][e] = (uint8_t)fx;
        if (!fx) loss_coeff(c->loss_mode, se / sw, ss / sw, c->dt, &c->ca[0][e], &c->cb[0][e]);
        else c->ca[0][e] = c->cb[0][e] = 0.0;
    }
    /* Ey(i,j,k): cells (i', j, k'), weight dx[i'] dz[k'] */
    for (int k = 0; k <= nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i <= nx; ++i) {
        double sw = 0, se = 0, ss = 0; int pec = 0;
        for (int kk = k - 1; kk <= k; ++kk) for (int ii = i - 1; ii <= i; ++ii) {
            if (ii < 0 || ii >= nx || kk < 0 || kk >= nz) continue;
            const int64_t q = CELL(ii, j, kk);
            double w = c->dx[ii] * c->dz[kk];
            sw += w; se += w * c->eps_c[q]; ss += w * c->sigma_c[q]; pec |= c->pec_c[q];
        }
        int fx = (i == 0 && wx0) || (i == nx && wx1) || (k == 0 && wz0) || (k == nz && wz1) || pec;
        int64_t e = EY(i, j, k);
        c->fixed[1][e] = (uint8_t)fx;
        if (!fx) loss_coeff(c->loss_mode, se / sw, ss / sw, c->dt, &c->ca[1][e], &c->cb[1][e]);
        else c->ca[1][e] = c->cb[1][e] = 0.0;
    }
    /* Ez(i,j,k): cells (i', j', k), weight dx[i'] dy[j'] */
    for (int k = 0; k < nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i <= nx; ++i) {
        double sw = 0, se = 0, ss = 0; int pec = 0;
        for (int jj = j - 1; jj <= j; ++jj) for (int ii = i - 1; ii <= i; ++ii) {
            if (ii < 0 || ii >= nx || jj < 0 || jj >= ny) continue;
            const int64_t q = CELL(ii, jj, k);
            double w = c->dx[ii] * c->dy[jj];
            sw += w; se += w * c->eps_c[q]; ss += w * c->sigma_c[q]; pec |= c->pec_c[q];
        }
        int fx = (i == 0 && wx0) || (i == nx && wx1) || (j == 0 && wy0) || (j == ny && wy1) || pec;
        int64_t e = EZ(i, j, k);
        c->fixed[2][e] = (uint8_t)fx;
        if (!fx) loss_coeff(c->loss_mode, se / sw, ss / sw, c->dt, &c->ca[2][e], &c->cb[2][e]);
        else c->ca[2][e] = c->cb[2][e] = 0.0;
    }
}

int32_t emo_create(const emo_grid *g, const uint8_t *mat_id, const emo_material *tab, int32_t n_mat,
                   double dt, emo_ctx **out) {
    if (!g || !mat_id || !tab || !out) return EMO_ERR_INVALID_ARG;
    if (g->nx < 1 || g->ny < 1 || g->nz < 1 || n_mat < 1 || n_mat > 256 || !(dt > 0.0)) return EMO_ERR_INVALID_ARG;
    if (g->loss_mode != EMO_LOSS_CD && g->loss_mode != EMO_LOSS_EXP) return EMO_ERR_INVALID_ARG;
    for (int b = 0; b < 6; ++b) if (g->bc[b] != EMO_BC_PEC && g->bc[b] != EMO_BC_PMC) return EMO_ERR_INVALID_ARG;
    for (int m = 0; m < n_mat; ++m)
        if (!(tab[m].eps > 0.0) || !(tab[m].mu > 0.0) || !(tab[m].sigma >= 0.0)) return EMO_ERR_INVALID_ARG;
    int nx = g->nx, ny = g->ny, nz = g->nz;
    for (int i = 0; i < nx; ++i) if (!(g->dx[i] > 0.0)) return EMO_ERR_INVALID_ARG;
    for (int j = 0; j < ny; ++j) if (!(g->dy[j] > 0.0)) return EMO_ERR_INVALID_ARG;
    for (int k = 0; k < nz; ++k) if (!(g->dz[k] > 0.0)) return EMO_ERR_INVALID_ARG;
    int64_t ncell = (int64_t)nx * ny * nz;
    for (int64_t c = 0; c < ncell; ++c) if (mat_id[c] >= n_mat) return EMO_ERR_INVALID_ARG;

    emo_ctx *c = (emo_ctx *)calloc(1, sizeof(emo_ctx));
    c->nx = nx; c->ny = ny; c->nz = nz; c->loss_mode = g->loss_mode; c->dt = dt;
    for (int b = 0; b < 6; ++b) c->bc[b] = g->bc[b];

    c->dx = (double *)malloc(sizeof(double) * nx); memcpy(c->dx, g->dx, sizeof(double) * nx);
    c->dy = (double *)malloc(sizeof(double) * ny); memcpy(c->dy, g->dy, sizeof(double) * ny);
    c->dz = (double *)malloc(sizeof(double) * nz); memcpy(c->dz, g->dz, sizeof(double) * nz);
    /* dual lengths: d~[i] = (d[i-1] + d[i])/2 inside, half a cell at the two ends */
    c->tx = (double *)malloc(sizeof(double) * (nx + 1));
    c->ty = (double *)malloc(sizeof(double) * (ny + 1));
    c->tz = (double *)malloc(sizeof(double) * (nz + 1));
    for (int i = 0; i <= nx; ++i) c->tx[i] = 0.5 * ((i > 0 ? c->dx[i - 1] : 0.0) + (i < nx ? c->dx[i] : 0.0));
    for (int j = 0; j <= ny; ++j) c->ty[j] = 0.5 * ((j > 0 ? c->dy[j - 1] : 0.0) + (j < ny ? c->dy[j] : 0.0));
    for (int k = 0; k <= nz; ++k) c->tz[k] = 0.5 * ((k > 0 ? c->dz[k - 1] : 0.0) + (k < nz ? c->dz[k] : 0.0));
    c->mat = (uint8_t *)malloc(ncell); memcpy(c->mat, mat_id, ncell);
    c->sigma_c = (double *)malloc(sizeof(double) * ncell);
    c->eps_c = (double *)malloc(sizeof(double) * ncell);
    c->pec_c = (uint8_t *)malloc(ncell);
    for (int64_t q = 0; q < ncell; ++q) {
        c->sigma_c[q] = tab[mat_id[q]].sigma; c->eps_c[q] = tab[mat_id[q]].eps; c->pec_c[q] = (uint8_t)(tab[mat_id[q]].flags & 1);
    }
    c->q = (double *)calloc(ncell, sizeof(double));
    for (int a = 0; a < 3; ++a) {
        int64_t ne = count_of(c, a), nf = count_of(c, 3 + a);
        c->E[a] = (double *)calloc(ne, sizeof(double));
        c->En[a] = (double *)calloc(ne, sizeof(double));
        c->J[a] = (double *)calloc(ne, sizeof(double));
        c->ca[a] = (double *)calloc(ne, sizeof(double));
        c->cb[a] = (double *)calloc(ne, sizeof(double));
        c->fixed[a] = (uint8_t *)calloc(ne, 1);
        c->H[a] = (double *)calloc(nf, sizeof(double));
        c->nu[a] = (double *)calloc(nf, sizeof(double));
    }

    edge_coefficients(c);
    /* ---- 1/mu on faces: length-weighted mean over the <=2 cells across the face ------------- */
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i <= nx; ++i) {
        double sw = 0, sn = 0;
        for (int ii = i - 1; ii <= i; ++ii) { if (ii < 0 || ii >= nx) continue;
            sw += c->dx[ii]; sn += c->dx[ii] / tab[mat_id[CELL(ii, j, k)]].mu; }
        c->nu[0][HX(i, j, k)] = sn / sw;
    }
    for (int k = 0; k < nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i < nx; ++i) {
        double sw = 0, sn = 0;
        for (int jj = j - 1; jj <= j; ++jj) { if (jj < 0 || jj >= ny) continue;
            sw += c->dy[jj]; sn += c->dy[jj] / tab[mat_id[CELL(i, jj, k)]].mu; }
        c->nu[1][HY(i, j, k)] = sn / sw;
    }
    for (int k = 0; k <= nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        double sw = 0, sn = 0;
        for (int kk = k - 1; kk <= k; ++kk) { if (kk < 0 || kk >= nz) continue;
            sw += c->dz[kk]; sn += c->dz[kk] / tab[mat_id[CELL(i, j, kk)]].mu; }
        c->nu[2][HZ(i, j, k)] = sn / sw;
    }
    *out = c;
    return EMO_OK;
}

static int edge_in_range(const emo_ctx *c, int comp, int i, int j, int k) {
    int sx, sy, sz; dims_of(c, comp, &sx, &sy, &sz);
    return i >= 0 && i < sx && j >= 0 && j < sy && k >= 0 && k < sz;
}

int32_t emo_set_source(emo_ctx *c, int32_t n_ports, const emo_port *ports, const emo_edge *edges,
                       int64_t n_edges, const double *wave, int64_t n_samples) {
    if (!c || n_ports < 0 || n_edges < 0 || n_samples < 0) return EMO_ERR_INVALID_ARG;
    int nx = c->nx, ny = c->ny; (void)nx; (void)ny;
    for (int64_t e = 0; e < n_edges; ++e) {
        if (edges[e].comp < 0 || edges[e].comp > 2) return EMO_ERR_INVALID_ARG;
        if (!edge_in_range(c, edges[e].comp, edges[e].i, edges[e].j, edges[e].k)) return EMO_ERR_INVALID_ARG;
        int sx, sy, sz; dims_of(c, edges[e].comp, &sx, &sy, &sz);
        if (c->fixed[edges[e].comp][IX(sx, sy, edges[e].i, edges[e].j, edges[e].k)]) return EMO_ERR_INVALID_ARG;
    }
    for (int p = 0; p < n_ports; ++p) {
        if (ports[p].edge_begin < 0 || ports[p].edge_end < ports[p].edge_begin || ports[p].edge_end > n_edges) return EMO_ERR_INVALID_ARG;
        if (ports[p].wave_offset < 0 || ports[p].wave_len < 0 || ports[p].wave_offset + ports[p].wave_len > n_samples) return EMO_ERR_INVALID_ARG;
    }
    free(c->ports); free(c->edges); free(c->wave);
    c->n_ports = n_ports; c->n_edges = n_edges; c->n_wave = n_samples;
    c->ports = (emo_port *)malloc(sizeof(emo_port) * (n_ports > 0 ? n_ports : 1));
    c->edges = (emo_edge *)malloc(sizeof(emo_edge) * (n_edges > 0 ? n_edges : 1));
    c->wave = (double *)malloc(sizeof(double) * (n_samples > 0 ? n_samples : 1));
    if (n_ports) memcpy(c->ports, ports, sizeof(emo_port) * n_ports);
    if (n_edges) memcpy(c->edges, edges, sizeof(emo_edge) * n_edges);
    if (n_samples) memcpy(c->wave, wave, sizeof(double) * n_samples);
    return EMO_OK;
}

int32_t emo_set_field(emo_ctx *c, int32_t comp, const double *src) {
    if (!c || comp < 0 || comp > 5 || !src) return EMO_ERR_INVALID_ARG;
    int64_t n = count_of(c, comp);
    if (comp < 3) {
        for (int64_t e = 0; e < n; ++e) c->E[comp][e] = c->fixed[comp][e] ? 0.0 : src[e];  /* PEC edges forced to 0 */
    } else memcpy(c->H[comp - 3], src, sizeof(double) * n);
    return EMO_OK;
}

int32_t emo_get_field(emo_ctx *c, int32_t comp, double *dst) {
    if (!c || comp < 0 || comp > 5 || !dst) return EMO_ERR_INVALID_ARG;
    memcpy(dst, comp < 3 ? c->E[comp] : c->H[comp - 3], sizeof(double) * count_of(c, comp));
    return EMO_OK;
}

/* Thermal stage (NEXT-1 of SURVEY.md 8(f); eq. (4)-(6), L84-L96), on the temperature RISE theta = T - T0
 * (M_kk annihilates constants and eq. (6) sees only T - T0, so T0 never enters):
 *   eq. (5)  theta^{n+1} = theta^n - dt/(rho c_p) (M_kk theta^n) + (dt P^{n+1})/(rho c_p)
 *   eq. (6)  sigma^{n+1} = sigma_0 / (1 + alpha theta^{n+1}),   then D_sigma(T^{n+1}) for the next E update (L78)
 * Readings (T1-T5): theta per CELL (the Joule heat is per cell, C7); dt P^{n+1} := the Joule energy density
 * dq_c this step deposited (time-centred, with the sigma(T^n) the E update used), so that EM loss == heat gained
 * exactly; M_kk = V0a^T D_k V0 as the cell-centred finite-volume -div k grad: the flux through the face between
 * cells c and c' is k_f A_f (theta_c - theta_c') / l~_f with the series (harmonic) conductivity
 * k_f l~_f^-1 = 2 / (d_c/k_c + d_c'/k_c'); no flux through the walls (adiabatic). */
static void thermal_step(emo_ctx *c) {
    const int nx = c->nx, ny = c->ny, nz = c->nz;
    const double dt = c->dt;
    const double *dx = c->dx, *dy = c->dy, *dz = c->dz, *th = c->theta, *kt = c->kth_c;
    int k;
#define COND(da, ka, db, kb) (((ka) > 0.0 && (kb) > 0.0) ? 2.0 / ((da) / (ka) + (db) / (kb)) : 0.0)   /* k_f / l~_f */
#pragma omp parallel for schedule(static)
    for (k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        const int64_t q = CELL(i, j, k);
        double out = 0.0;                               /* (M_kk theta)_c V_c : heat leaving cell c per second */
        if (i > 0)      out += COND(dx[i], kt[q], dx[i - 1], kt[CELL(i - 1, j, k)]) * dy[j] * dz[k] * (th[q] - th[CELL(i - 1, j, k)]);
        if (i < nx - 1) out += COND(dx[i], kt[q], dx[i + 1], kt[CELL(i + 1, j, k)]) * dy[j] * dz[k] * (th[q] - th[CELL(i + 1, j, k)]);
        if (j > 0)      out += COND(dy[j], kt[q], dy[j - 1], kt[CELL(i, j - 1, k)]) * dx[i] * dz[k] * (th[q] - th[CELL(i, j - 1, k)]);
        if (j < ny - 1) out += COND(dy[j], kt[q], dy[j + 1], kt[CELL(i, j + 1, k)]) * dx[i] * dz[k] * (th[q] - th[CELL(i, j + 1, k)]);
        if (k > 0)      out += COND(dz[k], kt[q], dz[k - 1], kt[CELL(i, j, k - 1)]) * dx[i] * dy[j] * (th[q] - th[CELL(i, j, k - 1)]);
        if (k < nz - 1) out += COND(dz[k], kt[q], dz[k + 1], kt[CELL(i, j, k + 1)]) * dx[i] * dy[j] * (th[q] - th[CELL(i, j, k + 1)]);
        const double vol = dx[i] * dy[j] * dz[k];
        c->theta_n[q] = th[q] - dt / c->rho_cp_c[q] * (out / vol) + c->dq[q] / c->rho_cp_c[q];
    }
#undef COND
    { double *t = c->theta; c->theta = c->theta_n; c->theta_n = t; }
    const int64_t ncell = (int64_t)nx * ny * nz;
    for (int64_t q = 0; q < ncell; ++q) c->sigma_c[q] = c->sigma0_c[q] / (1.0 + c->alpha_c[q] * c->theta[q]);   /* eq. (6) */
    edge_coefficients(c);                               /* D_sigma(T^{n+1}) for the next step */
}

/* ---- the NODAL thermal stage: the paper's placement of T (7 092 878 thermal unknowns = the nodes of its
 * 376 x 408 x 45 mesh) -- readings N1-N4 of DESIGN.md section 9, emo_set_thermal_nodal ----------------------------------
 *   N1  theta on the (nx+1)(ny+1)(nz+1) mesh nodes.
 *   N2  M_kk = V0a^T D_k V0 literally: V0 = node-to-edge difference over the edge length l_e (the negative
 *       gradient), D_k = diag(k_e A~_e) with k_e A~_e = sum over the <= 4 cells round the edge of k_c A_{c,e} / 4 (the
 *       area-weighted mean of C5 times the dual face, halved / quartered at the walls), V0a^T = the transposed
 *       incidence over the node's dual volume.  In heat units: C_n dtheta_n/dt = -sum_{e at n} (k_e A~_e / l_e)
 *       (theta_n - theta_m) + ..., C_n = sum over the <= 8 cells round the node of rho c_p V_c / 8.  No flux leaves
 *       the mesh (adiabatic, L142).
 *   N3  P_total = D_sigma e^2 (L86) is an EDGE vector: the energy the step dissipates on edge e,
 *       dQ_e = dt Ebar_e^2 l_e sum_{c round e} sigma_c(T^n) A_{c,e} / 4  (time-centred Ebar = (E^{n+1} + E^n)/2; summed
 *       over the edges this is exactly the dissipation of the discrete Poynting theorem and equals sum_c dq_c V_c of
 *       a4), goes half to each end node.
 *   N4  eq. (6) per cell with the mean of the cell's 8 node temperatures; everything else as T4. */
static double edge_cells_sum(const emo_ctx *c, int comp, int i, int j, int k, const double *val) {
    /* sum over the existing cells round edge (comp, i, j, k) of val_c * (cross-section of c normal to the edge) / 4 */
    const int nx = c->nx, ny = c->ny, nz = c->nz;
    double s = 0.0;
    for (int b = -1; b <= 0; ++b) for (int a = -1; a <= 0; ++a) {
        int ci = i, cj = j, ck = k; double area;
        if (comp == 0) { cj = j + a; ck = k + b; if (cj < 0 || cj >= ny || ck < 0 || ck >= nz) continue; area = c->dy[cj] * c->dz[ck]; }
        else if (comp == 1) { ci = i + a; ck = k + b; if (ci < 0 || ci >= nx || ck < 0 || ck >= nz) continue; area = c->dx[ci] * c->dz[ck]; }
        else { ci = i + a; cj = j + b; if (ci < 0 || ci >= nx || cj < 0 || cj >= ny) continue; area = c->dx[ci] * c->dy[cj]; }
        s += val[CELL(ci, cj, ck)] * area / 4.0;
    }
    return s;
}

static void thermal_step_nodal(emo_ctx *c) {
    const int nx = c->nx, ny = c->ny, nz = c->nz;
    const double dt = c->dt;
    const double *th = c->theta;
    /* after one_step swapped them, E holds E^{n+1} and En holds E^n */
#define NODE(i, j, k) IX(nx + 1, ny + 1, i, j, k)
    int k;
#pragma omp parallel for schedule(static)
    for (k = 0; k <= nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i <= nx; ++i) {
        double out = 0.0, heat = 0.0, cap = 0.0;
        /* the <= 6 edges at the node: (component, edge index, the node at its other end) */
        for (int comp = 0; comp < 3; ++comp) for (int side = -1; side <= 0; ++side) {
            int ei = i, ej = j, ek = k, mi = i, mj = j, mk = k; double len;
            if (comp == 0) { ei = i + side; mi = i + (side ? -1 : 1); if (ei < 0 || ei >= nx) continue; len = c->dx[ei]; }
            else if (comp == 1) { ej = j + side; mj = j + (side ? -1 : 1); if (ej < 0 || ej >= ny) continue; len = c->dy[ej]; }
            else { ek = k + side; mk = k + (side ? -1 : 1); if (ek < 0 || ek >= nz) continue; len = c->dz[ek]; }
            int sx, sy, sz; dims_of(c, comp, &sx, &sy, &sz);
            const int64_t e = IX(sx, sy, ei, ej, ek);
            out += edge_cells_sum(c, comp, ei, ej, ek, c->kth_c) / len * (th[NODE(i, j, k)] - th[NODE(mi, mj, mk)]);
            const double eb = 0.5 * (c->E[comp][e] + c->En[comp][e]);
            heat += 0.5 * dt * eb * eb * len * edge_cells_sum(c, comp, ei, ej, ek, c->sigma_c);
        }
        for (int dk = -1; dk <= 0; ++dk) for (int dj = -1; dj <= 0; ++dj) for (int di = -1; di <= 0; ++di) {
            const int ci = i + di, cj = j + dj, ck = k + dk;
            if (ci < 0 || ci >= nx || cj < 0 || cj >= ny || ck < 0 || ck >= nz) continue;
            cap += c->rho_cp_c[CELL(ci, cj, ck)] * c->dx[ci] * c->dy[cj] * c->dz[ck] / 8.0;
        }
        c->theta_n[NODE(i, j, k)] = th[NODE(i, j, k)] - dt * out / cap + heat / cap;
    }
    { double *t = c->theta; c->theta = c->theta_n; c->theta_n = t; }
    for (k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        double m = 0.0;
        for (int dk = 0; dk <= 1; ++dk) for (int dj = 0; dj <= 1; ++dj) for (int di = 0; di <= 1; ++di) m += c->theta[NODE(i + di, j + dj, k + dk)];
        c->sigma_c[CELL(i, j, k)] = c->sigma0_c[CELL(i, j, k)] / (1.0 + c->alpha_c[CELL(i, j, k)] * (m / 8.0));      /* eq. (6) */
    }
#undef NODE
    edge_coefficients(c);
}

/* One step n -> n+1 (SURVEY.md 8(c) "One step"): a1 H update, a3 source, a2 E update, a4 Joule. */
static void one_step(emo_ctx *c) {
    const int nx = c->nx, ny = c->ny, nz = c->nz;
    const double dt = c->dt;
    const double *dx = c->dx, *dy = c->dy, *dz = c->dz, *tx = c->tx, *ty = c->ty, *tz = c->tz;
    double *Ex = c->E[0], *Ey = c->E[1], *Ez = c->E[2];
    double *Hx = c->H[0], *Hy = c->H[1], *Hz = c->H[2];
    int k;

    /* a1: H^{n+1/2} = H^{n-1/2} - dt nu (C_e E^n) */
#pragma omp parallel for schedule(static)
    for (k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i <= nx; ++i)
        Hx[HX(i, j, k)] -= dt * c->nu[0][HX(i, j, k)] *
            ((Ez[EZ(i, j + 1, k)] - Ez[EZ(i, j, k)]) / dy[j] - (Ey[EY(i, j, k + 1)] - Ey[EY(i, j, k)]) / dz[k]);
#pragma omp parallel for schedule(static)
    for (k = 0; k < nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i < nx; ++i)
        Hy[HY(i, j, k)] -= dt * c->nu[1][HY(i, j, k)] *
            ((Ex[EX(i, j, k + 1)] - Ex[EX(i, j, k)]) / dz[k] - (Ez[EZ(i + 1, j, k)] - Ez[EZ(i, j, k)]) / dx[i]);
#pragma omp parallel for schedule(static)
    for (k = 0; k <= nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i)
        Hz[HZ(i, j, k)] -= dt * c->nu[2][HZ(i, j, k)] *
            ((Ey[EY(i + 1, j, k)] - Ey[EY(i, j, k)]) / dx[i] - (Ex[EX(i, j + 1, k)] - Ex[EX(i, j, k)]) / dy[j]);

    /* a3: J(e) = sum over ports of amplitude * weight * wave[n]  (0 beyond the table) */
    for (int p = 0; p < c->n_ports; ++p) {
        const emo_port *pt = &c->ports[p];
        double w = (c->step < pt->wave_len) ? c->wave[pt->wave_offset + c->step] : 0.0;
        for (int64_t e = pt->edge_begin; e < pt->edge_end; ++e) {
            const emo_edge *ed = &c->edges[e];
            int sx, sy, sz; dims_of(c, ed->comp, &sx, &sy, &sz);
            c->J[ed->comp][IX(sx, sy, ed->i, ed->j, ed->k)] += pt->amplitude * ed->weight * w;
        }
    }

    /* a2: E^{n+1} = ca E^n + cb (C_h H^{n+1/2} - J^{n+1/2}) on every non-fixed edge.
     * H with an out-of-range index is 0; only reachable from the non-fixed edges of a PMC wall, where
     * the dual length ty/tz/tx is the half cell (SURVEY.md 8(c) "One step" a2, C8). */
#define HXG(i, j, k) (((j) >= 0 && (j) < ny && (k) >= 0 && (k) < nz) ? Hx[HX(i, j, k)] : 0.0)
#define HYG(i, j, k) (((i) >= 0 && (i) < nx && (k) >= 0 && (k) < nz) ? Hy[HY(i, j, k)] : 0.0)
#define HZG(i, j, k) (((i) >= 0 && (i) < nx && (j) >= 0 && (j) < ny) ? Hz[HZ(i, j, k)] : 0.0)
    double *Exn = c->En[0], *Eyn = c->En[1], *Ezn = c->En[2];
#pragma omp parallel for schedule(static)
    for (k = 0; k <= nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i < nx; ++i) {
        int64_t e = EX(i, j, k);
        if (c->fixed[0][e]) { Exn[e] = 0.0; continue; }
        Exn[e] = c->ca[0][e] * Ex[e] + c->cb[0][e] *
            ((HZG(i, j, k) - HZG(i, j - 1, k)) / ty[j] - (HYG(i, j, k) - HYG(i, j, k - 1)) / tz[k] - c->J[0][e]);
    }
#pragma omp parallel for schedule(static)
    for (k = 0; k <= nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i <= nx; ++i) {
        int64_t e = EY(i, j, k);
        if (c->fixed[1][e]) { Eyn[e] = 0.0; continue; }
        Eyn[e] = c->ca[1][e] * Ey[e] + c->cb[1][e] *
            ((HXG(i, j, k) - HXG(i, j, k - 1)) / tz[k] - (HZG(i, j, k) - HZG(i - 1, j, k)) / tx[i] - c->J[1][e]);
    }
#pragma omp parallel for schedule(static)
    for (k = 0; k < nz; ++k) for (int j = 0; j <= ny; ++j) for (int i = 0; i <= nx; ++i) {
        int64_t e = EZ(i, j, k);
        if (c->fixed[2][e]) { Ezn[e] = 0.0; continue; }
        Ezn[e] = c->ca[2][e] * Ez[e] + c->cb[2][e] *
            ((HYG(i, j, k) - HYG(i - 1, j, k)) / tx[i] - (HXG(i, j, k) - HXG(i, j - 1, k)) / ty[j] - c->J[2][e]);
    }

#undef HXG
#undef HYG
#undef HZG

    /* a4: q_c += dt sigma_c * 1/4 sum over the 12 edges of c of ((E^{n+1} + E^n)/2)^2 */
#define B2(A, An, idx) ({ double b_ = 0.5 * ((An)[idx] + (A)[idx]); b_ * b_; })
#pragma omp parallel for schedule(static)
    for (k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
        double s = 0.25 * (
            B2(Ex, Exn, EX(i, j, k)) + B2(Ex, Exn, EX(i, j + 1, k)) + B2(Ex, Exn, EX(i, j, k + 1)) + B2(Ex, Exn, EX(i, j + 1, k + 1)) +
            B2(Ey, Eyn, EY(i, j, k)) + B2(Ey, Eyn, EY(i + 1, j, k)) + B2(Ey, Eyn, EY(i, j, k + 1)) + B2(Ey, Eyn, EY(i + 1, j, k + 1)) +
            B2(Ez, Ezn, EZ(i, j, k)) + B2(Ez, Ezn, EZ(i + 1, j, k)) + B2(Ez, Ezn, EZ(i, j + 1, k)) + B2(Ez, Ezn, EZ(i + 1, j + 1, k)));
        const double dq = dt * c->sigma_c[CELL(i, j, k)] * s;     /* heat deposited in this step, sigma = sigma(T^n) */
        c->q[CELL(i, j, k)] += dq;
        if (c->thermal) c->dq[CELL(i, j, k)] = dq;
    }
#undef B2

    /* E <- E^{n+1}; clear the source scatter */
    for (int a = 0; a < 3; ++a) { double *t = c->E[a]; c->E[a] = c->En[a]; c->En[a] = t; }
    for (int p = 0; p < c->n_ports; ++p) {
        const emo_port *pt = &c->ports[p];
        for (int64_t e = pt->edge_begin; e < pt->edge_end; ++e) {
            const emo_edge *ed = &c->edges[e];
            int sx, sy, sz; dims_of(c, ed->comp, &sx, &sy, &sz);
            c->J[ed->comp][IX(sx, sy, ed->i, ed->j, ed->k)] = 0.0;
        }
    }
    if (c->thermal == 1) thermal_step(c);
    if (c->thermal == 2) thermal_step_nodal(c);
    c->step += 1;
}

int32_t emo_step(emo_ctx *c, int64_t n) {
    if (!c || n < 0) return EMO_ERR_INVALID_ARG;
    for (int64_t s = 0; s < n; ++s) one_step(c);
    return EMO_OK;
}

/* Joule outputs (SURVEY.md 8(b) em_joule): instantaneous p_c = sigma_c 1/4 sum_12 (E_e^n)^2
 * (paper-literal D_sigma e^2), accumulated q_c, total Q = sum_c q_c V_c (Kahan). */
int32_t emo_joule(emo_ctx *c, double *power_density, double *energy_density, double *total_energy, int32_t reset) {
    if (!c) return EMO_ERR_INVALID_ARG;
    const int nx = c->nx, ny = c->ny, nz = c->nz;
    const double *Ex = c->E[0], *Ey = c->E[1], *Ez = c->E[2];
#define SQ(A, idx) ((A)[idx] * (A)[idx])
    if (power_density)
        for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
            double s = 0.25 * (
                SQ(Ex, EX(i, j, k)) + SQ(Ex, EX(i, j + 1, k)) + SQ(Ex, EX(i, j, k + 1)) + SQ(Ex, EX(i, j + 1, k + 1)) +
                SQ(Ey, EY(i, j, k)) + SQ(Ey, EY(i + 1, j, k)) + SQ(Ey, EY(i, j, k + 1)) + SQ(Ey, EY(i + 1, j, k + 1)) +
                SQ(Ez, EZ(i, j, k)) + SQ(Ez, EZ(i + 1, j, k)) + SQ(Ez, EZ(i, j + 1, k)) + SQ(Ez, EZ(i + 1, j + 1, k)));
            power_density[CELL(i, j, k)] = c->sigma_c[CELL(i, j, k)] * s;
        }
#undef SQ
    int64_t ncell = (int64_t)nx * ny * nz;
    if (energy_density) memcpy(energy_density, c->q, sizeof(double) * ncell);
    if (total_energy) {
        double sum = 0.0, comp = 0.0;
        for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
            double v = c->q[CELL(i, j, k)] * (c->dx[i] * c->dy[j] * c->dz[k]);
            double y = v - comp, t = sum + y;
            comp = (t - sum) - y; sum = t;
        }
        *total_energy = sum;
    }
    if (reset) memset(c->q, 0, sizeof(double) * ncell);
    return EMO_OK;
}

int32_t emo_probe(emo_ctx *c, int32_t n_pts, const emo_probe_pt *pts, double *out) {
    if (!c || n_pts < 0 || (n_pts && (!pts || !out))) return EMO_ERR_INVALID_ARG;
    for (int p = 0; p < n_pts; ++p) {
        int comp = pts[p].comp;
        if (comp < 0 || comp > 5 || !edge_in_range(c, comp, pts[p].i, pts[p].j, pts[p].k)) return EMO_ERR_INVALID_ARG;
        int sx, sy, sz; dims_of(c, comp, &sx, &sy, &sz);
        const double *a = comp < 3 ? c->E[comp] : c->H[comp - 3];
        out[p] = a[IX(sx, sy, pts[p].i, pts[p].j, pts[p].k)];
    }
    return EMO_OK;
}

int32_t emo_reset(emo_ctx *c) {
    if (!c) return EMO_ERR_INVALID_ARG;
    for (int a = 0; a < 3; ++a) {
        memset(c->E[a], 0, sizeof(double) * count_of(c, a));
        memset(c->En[a], 0, sizeof(double) * count_of(c, a));
        memset(c->H[a], 0, sizeof(double) * count_of(c, 3 + a));
    }
    memset(c->q, 0, sizeof(double) * (int64_t)c->nx * c->ny * c->nz);
    if (c->thermal) {
        const int64_t ncell = (int64_t)c->nx * c->ny * c->nz;
        memset(c->theta, 0, sizeof(double) * (c->thermal == 2 ? (int64_t)(c->nx + 1) * (c->ny + 1) * (c->nz + 1) : ncell));
        memcpy(c->sigma_c, c->sigma0_c, sizeof(double) * ncell);
        edge_coefficients(c);
    }
    c->step = 0;
    return EMO_OK;
}

int64_t emo_step_index(const emo_ctx *c) { return c ? c->step : -1; }

/* ---- thermal coupling API (NEXT-1) ---------------------------------------------------------------------------- */
typedef struct { double rho_cp, k, alpha; } emo_thermal_material;   /* J/(m^3 K), W/(m K), 1/K */

/* Switches the coupling on: per-material volumetric heat capacity, thermal conductivity and temperature coefficient
 * of resistance; theta = 0, sigma = sigma_0 (the table's).  rho_cp > 0, k >= 0 (0 = no conduction through the cell). */
static int32_t set_thermal_placed(emo_ctx *c, const emo_thermal_material *tt, int32_t n_mat, int32_t placement) {
    if (!c || !tt || n_mat < 1) return EMO_ERR_INVALID_ARG;
    if (c->thermal && c->thermal != placement) return EMO_ERR_INVALID_ARG;      /* one placement per context */
    const int64_t ncell = (int64_t)c->nx * c->ny * c->nz;
    const int64_t nth = placement == 2 ? (int64_t)(c->nx + 1) * (c->ny + 1) * (c->nz + 1) : ncell;
    for (int64_t q = 0; q < ncell; ++q) if (c->mat[q] >= n_mat) return EMO_ERR_INVALID_ARG;
    for (int m = 0; m < n_mat; ++m) if (!(tt[m].rho_cp > 0.0) || !(tt[m].k >= 0.0)) return EMO_ERR_INVALID_ARG;
    if (!c->thermal) {
        c->theta = (double *)calloc(nth, sizeof(double)); c->theta_n = (double *)calloc(nth, sizeof(double));
        c->dq = (double *)calloc(ncell, sizeof(double));
        c->sigma0_c = (double *)malloc(sizeof(double) * ncell); c->rho_cp_c = (double *)malloc(sizeof(double) * ncell);
        c->kth_c = (double *)malloc(sizeof(double) * ncell); c->alpha_c = (double *)malloc(sizeof(double) * ncell);
        memcpy(c->sigma0_c, c->sigma_c, sizeof(double) * ncell);
        c->thermal = placement;
    }
    for (int64_t q = 0; q < ncell; ++q) {
        c->rho_cp_c[q] = tt[c->mat[q]].rho_cp; c->kth_c[q] = tt[c->mat[q]].k; c->alpha_c[q] = tt[c->mat[q]].alpha;
        c->sigma_c[q] = c->sigma0_c[q];
    }
    memset(c->theta, 0, sizeof(double) * nth);
    edge_coefficients(c);
    return EMO_OK;
}
int32_t emo_set_thermal(emo_ctx *c, const emo_thermal_material *tt, int32_t n_mat) { return set_thermal_placed(c, tt, n_mat, 1); }
/* the same with theta on the mesh NODES (the paper's placement; thermal_step_nodal above) */
int32_t emo_set_thermal_nodal(emo_ctx *c, const emo_thermal_material *tt, int32_t n_mat) { return set_thermal_placed(c, tt, n_mat, 2); }
/* number of temperature unknowns: cells (placement 1) or nodes (2); 0 if the coupling is off */
int64_t emo_thermal_unknowns(const emo_ctx *c) {
    if (!c || !c->thermal) return 0;
    return c->thermal == 2 ? (int64_t)(c->nx + 1) * (c->ny + 1) * (c->nz + 1) : (int64_t)c->nx * c->ny * c->nz;
}

int32_t emo_get_temperature_rise(emo_ctx *c, double *dst) {
    if (!c || !dst || !c->thermal) return EMO_ERR_INVALID_ARG;
    memcpy(dst, c->theta, sizeof(double) * emo_thermal_unknowns(c));
    return EMO_OK;
}

/* sets theta and refreshes sigma(T) (eq. 6) and the edge coefficients */
int32_t emo_set_temperature_rise(emo_ctx *c, const double *src) {
    if (!c || !src || !c->thermal) return EMO_ERR_INVALID_ARG;
    const int64_t ncell = (int64_t)c->nx * c->ny * c->nz;
    if (c->thermal == 2) {                    /* nodal: sigma(T) from the mean of the cell's 8 node temperatures (N4) */
        const int nx = c->nx, ny = c->ny, nz = c->nz;
        memcpy(c->theta, src, sizeof(double) * emo_thermal_unknowns(c));
        for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
            double m = 0.0;
            for (int dk = 0; dk <= 1; ++dk) for (int dj = 0; dj <= 1; ++dj) for (int di = 0; di <= 1; ++di)
                m += c->theta[IX(nx + 1, ny + 1, i + di, j + dj, k + dk)];
            if (!(1.0 + c->alpha_c[CELL(i, j, k)] * (m / 8.0) > 0.0)) return EMO_ERR_INVALID_ARG;
            c->sigma_c[CELL(i, j, k)] = c->sigma0_c[CELL(i, j, k)] / (1.0 + c->alpha_c[CELL(i, j, k)] * (m / 8.0));
        }
        edge_coefficients(c);
        return EMO_OK;
    }
    for (int64_t q = 0; q < ncell; ++q) if (!(1.0 + c->alpha_c[q] * src[q] > 0.0)) return EMO_ERR_INVALID_ARG;
    memcpy(c->theta, src, sizeof(double) * ncell);
    for (int64_t q = 0; q < ncell; ++q) c->sigma_c[q] = c->sigma0_c[q] / (1.0 + c->alpha_c[q] * c->theta[q]);
    edge_coefficients(c);
    return EMO_OK;
}
